// lm_handle.cuh -- the solver handle of liblm: pair-kernel variants, NCCL loader, state, error helpers and the launch chooser.
// Included by lm_api.cu only (one translation unit); everything after the handle lives in an anonymous namespace.
#pragma once

namespace lm {

// ---------------------------------------------------------------- pair-kernel variants
// LARGE: 256 threads x TPT targets (TPT/2 packed pairs per thread), tiles of up to 512 sources.
// SMALL: 64 x 2, tiles of up to 64 sources (fills 148 SMs when N is small, SURVEY.md sec. 7 "Small N").
// SUB = sources per overlap-vote chunk = the unit in which sources are dealt to the j-splits;
// npad is a multiple of NPAD_QUANTUM, which every SUB divides.
constexpr int NPAD_QUANTUM = 32;
constexpr int L_BLOCK = 256, L_TJ = 512, L_STAGES = 2;
constexpr int S_BLOCK = 64, S_TPT = 2, S_TJ = 64, S_STAGES = 2;
constexpr int64_t MAX_SOURCES_PER_CTA = 262144;   // bounds the top level of the two-level fp32 summation

template <typename T> struct Variant {
    void (*kernel)(const PairParams<T>);
    int nrhs, ang, block, tpt, tj, sub, smem;
    int ctas_per_sm;      // filled at first use (occupancy API)
    double efficiency;    // relative per-pair throughput used by the launch chooser
    int wall;             // 1: the single-wall variant (free-space pair + wall correction)
    int acc64;            // 1: fp32 pair math with fp64 accumulation (LM_OPT_ACCUMULATE_F64)
};

template <typename T, int NRHS, bool ANG, int TPT, int SUB, int MINB, bool WALL = false, bool ACC64 = false> Variant<T> make_large()
{
    using Tr = PairKernelTraits<T, NRHS, ANG, TPT, L_BLOCK, L_TJ, L_STAGES, SUB, ACC64>;
    static_assert(NPAD_QUANTUM % SUB == 0, "every SUB divides NPAD_QUANTUM");
    return {rpy_pair_kernel<T, NRHS, ANG, TPT, L_BLOCK, L_TJ, L_STAGES, SUB, MINB, WALL, ACC64>, NRHS, ANG, L_BLOCK, TPT, L_TJ, SUB, Tr::SMEM_BYTES, 0, 1.0, WALL, ACC64};
}
template <typename T, int NRHS, bool ANG, int SUB, int MINB, bool WALL = false> Variant<T> make_small()
{
    using Tr = PairKernelTraits<T, NRHS, ANG, S_TPT, S_BLOCK, S_TJ, S_STAGES, SUB>;
    static_assert(NPAD_QUANTUM % SUB == 0, "every SUB divides NPAD_QUANTUM");
    return {rpy_pair_kernel<T, NRHS, ANG, S_TPT, S_BLOCK, S_TJ, S_STAGES, SUB, MINB, WALL>, NRHS, ANG, S_BLOCK, S_TPT, S_TJ, SUB, Tr::SMEM_BYTES, 0, 0.8, WALL, 0};
}

template <typename T> std::vector<Variant<T>> build_variants();
template <> std::vector<Variant<float>> build_variants<float>()
{
    return {make_large<float, 1, false, 4, 32, 2>(), make_large<float, 2, false, 4, 32, 1>(), make_large<float, 4, false, 4, 32, 1>(),
            make_large<float, 1, true, 2, 32, 2>(),  make_large<float, 2, true, 2, 32, 1>(),
            make_small<float, 1, false, 32, 8>(), make_small<float, 2, false, 32, 8>(), make_small<float, 4, false, 32, 6>(),
            make_small<float, 1, true, 32, 8>(),  make_small<float, 2, true, 32, 6>(),
            // single wall (the wall correction roughly triples the per-pair work and the live registers)
            make_large<float, 1, false, 2, 32, 2, true>(), make_large<float, 2, false, 2, 32, 1, true>(),
            make_large<float, 1, true, 2, 32, 1, true>(),  make_large<float, 2, true, 2, 32, 1, true>(),
            make_small<float, 1, false, 32, 6, true>(), make_small<float, 2, false, 32, 6, true>(),
            make_small<float, 1, true, 32, 4, true>(),  make_small<float, 2, true, 32, 4, true>(),
            // fp32 pair math, fp64 accumulation (LARGE shape only: the option is for large sums; any N is still served)
            make_large<float, 1, false, 4, 32, 2, false, true>(), make_large<float, 2, false, 4, 32, 1, false, true>(), make_large<float, 4, false, 4, 32, 1, false, true>(),
            make_large<float, 1, true, 2, 32, 2, false, true>(),  make_large<float, 2, true, 2, 32, 1, false, true>(),
            make_large<float, 1, false, 2, 32, 2, true, true>(), make_large<float, 2, false, 2, 32, 1, true, true>(),
            make_large<float, 1, true, 2, 32, 1, true, true>(),  make_large<float, 2, true, 2, 32, 1, true, true>()};
}
template <> std::vector<Variant<double>> build_variants<double>()
{
    return {make_large<double, 1, false, 4, 32, 1>(), make_large<double, 2, false, 2, 32, 1>(), make_large<double, 4, false, 2, 32, 1>(),
            make_large<double, 1, true, 2, 32, 1>(),  make_large<double, 2, true, 2, 32, 1>(),
            make_small<double, 1, false, 32, 8>(), make_small<double, 2, false, 32, 6>(), make_small<double, 4, false, 32, 4>(),
            make_small<double, 1, true, 32, 6>(),  make_small<double, 2, true, 32, 4>(),
            make_large<double, 1, false, 2, 32, 1, true>(), make_large<double, 2, false, 2, 32, 1, true>(),
            make_large<double, 1, true, 2, 32, 1, true>(),  make_large<double, 2, true, 2, 32, 1, true>(),
            make_small<double, 1, false, 32, 4, true>(), make_small<double, 2, false, 32, 4, true>(),
            make_small<double, 1, true, 32, 3, true>(),  make_small<double, 2, true, 32, 2, true>()};
}

struct LaunchPlan {
    int variant = -1;
    int i_tiles = 0, j_splits = 0, n_units = 0;
};

// ---------------------------------------------------------------- one-launch small-N kernel (rpy_small.cuh)
template <typename T> struct SmallVariant {
    void (*kernel)(const SmallParams<T>);
    int nrhs, ang, wall;
    size_t (*smem)(int warps, int src_per_warp);
};
template <typename T, int NRHS, bool ANG, bool WALL> SmallVariant<T> make_fused()
{
    return {rpy_small_kernel<T, NRHS, ANG, WALL>, NRHS, ANG, WALL, small_smem_bytes<T, NRHS, ANG>};
}
template <typename T> std::vector<SmallVariant<T>> build_small_variants()
{
    return {make_fused<T, 1, false, false>(), make_fused<T, 2, false, false>(), make_fused<T, 4, false, false>(),
            make_fused<T, 1, true, false>(),  make_fused<T, 2, true, false>(),
            make_fused<T, 1, false, true>(),  make_fused<T, 2, false, true>(),
            make_fused<T, 1, true, true>(),   make_fused<T, 2, true, true>()};
}
constexpr size_t SMALL_MAX_SMEM = 96 * 1024;      // dynamic shared memory the small kernel may ask for

struct SmallPlan {
    int variant = -1;
    int i_tiles = 0, cluster = 0, warps = 0, src_per_warp = 0;
    size_t smem = 0;
};

}  // namespace lm

// ---------------------------------------------------------------- NCCL, loaded at run time (row-sharded applies only)
// The library does not link NCCL: a single-GPU user never needs it.  lm_dist_* resolve the few entry
// points below from the libnccl already in the process (PyTorch's) or, failing that, the system one.
namespace lm {
struct NcclApi {
    struct UniqueId { char internal[128]; };
    typedef void* Comm;
    int (*GetUniqueId)(UniqueId*) = nullptr;
    int (*CommInitRank)(Comm*, int, UniqueId, int) = nullptr;
    int (*CommDestroy)(Comm) = nullptr;
    int (*AllGather)(const void*, void*, size_t, int, Comm, cudaStream_t) = nullptr;
    int (*Broadcast)(const void*, void*, size_t, int, int, Comm, cudaStream_t) = nullptr;
    int (*AllReduce)(const void*, void*, size_t, int, int, Comm, cudaStream_t) = nullptr;
    int (*GroupStart)() = nullptr;
    int (*GroupEnd)() = nullptr;
    const char* (*GetErrorString)(int) = nullptr;
    bool ok = false;
    std::string why;
};
constexpr int NCCL_INT32 = 2, NCCL_FLOAT32 = 7, NCCL_FLOAT64 = 8;   // ncclDataType_t values (nccl.h)
constexpr int NCCL_MAX = 2;                                          // ncclRedOp_t value (nccl.h: ncclSum, ncclProd, ncclMax, ...)

inline NcclApi& nccl_api()
{
    static NcclApi api;
    static bool tried = false;
    if (tried) return api;
    tried = true;
    void* lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_NOLOAD);
    if (!lib) lib = dlopen("libnccl.so.2", RTLD_NOW | RTLD_GLOBAL);
    if (!lib) { api.why = std::string("cannot load libnccl.so.2: ") + dlerror(); return api; }
    auto sym = [&](const char* name) { void* p = dlsym(lib, name); if (!p) api.why = std::string("libnccl.so.2 lacks ") + name; return p; };
    api.GetUniqueId = (int (*)(NcclApi::UniqueId*))sym("ncclGetUniqueId");
    api.CommInitRank = (int (*)(NcclApi::Comm*, int, NcclApi::UniqueId, int))sym("ncclCommInitRank");
    api.CommDestroy = (int (*)(NcclApi::Comm))sym("ncclCommDestroy");
    api.AllGather = (int (*)(const void*, void*, size_t, int, NcclApi::Comm, cudaStream_t))sym("ncclAllGather");
    api.Broadcast = (int (*)(const void*, void*, size_t, int, int, NcclApi::Comm, cudaStream_t))sym("ncclBroadcast");
    api.AllReduce = (int (*)(const void*, void*, size_t, int, int, NcclApi::Comm, cudaStream_t))sym("ncclAllReduce");
    api.GroupStart = (int (*)())sym("ncclGroupStart");
    api.GroupEnd = (int (*)())sym("ncclGroupEnd");
    api.GetErrorString = (const char* (*)(int))sym("ncclGetErrorString");
    api.ok = api.GetUniqueId && api.CommInitRank && api.CommDestroy && api.AllGather && api.Broadcast && api.AllReduce && api.GroupStart && api.GroupEnd && api.GetErrorString;
    return api;
}
}  // namespace lm

using namespace lm;

// ---------------------------------------------------------------- handle
struct lm_solver {
    int precision = LM_F32;
    int64_t N = 0, npad = 0;
    double eta = 1.0, a = 1.0;
    double len_scale = 1.0;    // power of two nearest 1/a: lengths are stored x len_scale, so the kernels see a radius in [0.71, 1.41]
    int angular = 0;
    int wall = 0;              // geometry ("open","open","single_wall"): lm_set_wall
    double wall_z = 0.0;       // the wall is the plane z = wall_z, fluid above (the paper's setParameters(wallHeight))
    int max_iter = 100;
    int lz_rule = lm::RULE_ESTIMATE;   // Lanczos stopping rule (reading S3; LM_OPT_LANCZOS_RULE)
    bool graph_replay = true;          // short applies / Lanczos iterations replayed as CUDA graphs (LM_OPT_GRAPH_REPLAY)
    bool share_first_apply = true;     // M.[F;T] rides along with the first Lanczos apply (LM_OPT_SHARE_FIRST_APPLY)
    int device = 0, sm_count = 0;
    bool have_pos = false;
    std::string err;
    int last_iters = -1;

    void* pos_soa = nullptr;
    void* vec_soa = nullptr;   size_t vec_soa_bytes = 0;
    void* partial = nullptr;   size_t partial_bytes = 0;

    // Lanczos workspace
    void* V = nullptr;         size_t V_bytes = 0;
    void* w = nullptr;         size_t w_bytes = 0;
    double* d_scal = nullptr;  // [0] |z|^2  [1] alpha  [2] beta^2
    double* d_block = nullptr; // block partials of the reductions
    unsigned int* d_ticket = nullptr;
    int* d_newest = nullptr;   // index of the newest basis vector (read by the iteration's kernels)
    double* d_coef = nullptr;  size_t coef_cap = 0;   // coef_cap also sizes the buffers below
    double* d_gram_part = nullptr;
    // mapped pinned host memory the kernels write the stopping-test scalars into
    double* h_ab = nullptr;    // [1] |z|^2; [2k], [2k+1]: alpha_k, beta_k^2
    double* h_gram = nullptr;  // column c at [c * (max_iter + 2) + j] = V[j].V[c], j <= c
    cudaEvent_t lz_ev[2] = {nullptr, nullptr};   // iteration k's scalars have landed (parity k & 1)
    std::vector<lm::LanczosStopper> lz_stop;     // host state of the last Lanczos call, one per noise vector (lm_lanczos_history)
    unsigned *d_word = nullptr, *h_word = nullptr;   // the stopping verdicts rank 0 broadcasts (row-sharded runs)
    // one Lanczos iteration captured as a CUDA graph (small N: the loop is launch-bound)
    cudaStream_t cap_stream = nullptr;
    cudaGraphExec_t lz_graph = nullptr;
    struct GraphKey { const void *V, *w, *vec, *partial, *pos; int kmax, variant, splits, prec; } lz_key = {nullptr, nullptr, nullptr, nullptr, nullptr, 0, 0, 0, 0};

    // Brownian-dynamics step (lm_bd_step): F, v_n, v_{n-1}, noise velocity, angular scratch x2, position staging
    // [7], [8]: the drift sample (linear, angular) of a step with a random-finite-difference term
    void* bd[9] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    size_t bd_bytes[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool bd_have_prev = false;
    bool steric_attr_set = false;
    // random finite difference (lm_thermal_drift_rfd): displaced packed positions, U(X-) linear / angular
    void* rfd[3] = {nullptr, nullptr, nullptr};
    size_t rfd_bytes[3] = {0, 0, 0};

    // row-sharded applies over NCCL (lm_dist_init): rank r computes target rows [r B, min((r+1) B, N)), B = rows_per_rank
    int dist_ranks = 0, dist_rank = 0;        // dist_ranks == 0: not distributed
    int64_t rows_per_rank = 0;
    void* nccl_comm = nullptr;
    void* gath[2 * MAX_RHS] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   // all-gather buffers, 3 B ranks each
    size_t gath_bytes[2 * MAX_RHS] = {0, 0, 0, 0, 0, 0, 0, 0};
    int64_t row_begin = 0, row_end = 0;       // the target rows every apply computes ([0, N) unless sharded / lm_mdot_rows)

    // staging for the _host entry points
    void* st[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};  // pos, f, t, noise, lin, ang
    size_t st_bytes[6] = {0, 0, 0, 0, 0, 0};

    // variants (typed; only the handle's precision is populated)
    std::vector<Variant<float>> vf;
    std::vector<Variant<double>> vd;
    std::vector<SmallVariant<float>> sf;
    std::vector<SmallVariant<double>> sd;
    // one-launch small-N kernel (LM_OPT_SMALL_KERNEL): 1 = where the launch chooser prefers it, 0 = never,
    // (cluster << 8 | warps) = always, with that shape (plan sweeps)
    int small_kernel = 1;
    int max_cluster = 1;       // largest cluster size (<= 8) the device can co-schedule for the one-launch kernel (occupancy API, at lm_create)
    bool acc64 = false;             // LM_OPT_ACCUMULATE_F64 (fp32 handles): fp64 accumulation of the fp32 pair terms
    bool gather_in_caller = true;   // LM_OPT_GATHER_IN_PLACE: row-sharded applies all-gather straight into the caller's arrays when the blocks tile [0, N)
    int force_splits = 0;      // LM_OPT_J_SPLITS: > 0 fixes the number of j-splits of the general path (plan sweeps)
    struct SmallSlot { bool valid = false; int64_t rb = 0, re = 0; int mode = 0; lm::SmallPlan plan; } small_cache[lm::MAX_RHS + 1];

    // launch plans are pure functions of (nrhs, row range): cached, the chooser's search is off the per-call path
    struct PlanSlot { bool valid = false; int64_t rb = 0, re = 0; lm::LaunchPlan plan; } plan_cache[lm::MAX_RHS + 1];

    // small-N applies (pack + pair kernel + reduce) replayed as a CUDA graph when called again with the same buffers
    struct ApplyKey {
        const void *f[lm::MAX_RHS], *t[lm::MAX_RHS], *lin[lm::MAX_RHS], *ang[lm::MAX_RHS];
        const void *pos, *vec, *partial;
        int64_t rb, re;
        int nrhs, variant, splits, pad;
    };
    struct ApplySlot { bool have_last = false; ApplyKey last, graph_key; cudaGraphExec_t exec = nullptr; } apply_graph[lm::MAX_RHS + 1];

    // stats
    int64_t n_pair = 0, n_aux = 0;
    double pairs = 0.0, pair_ms = 0.0;
    bool profiling = false;
    std::vector<std::pair<cudaEvent_t, cudaEvent_t>> pending;
    std::vector<cudaEvent_t> event_pool;
};

namespace {

int fail(lm_solver* h, int code, const std::string& msg)
{
    if (h) h->err = msg;
    return code;
}

#define LM_CUDA(h, expr)                                                                              \
    do {                                                                                              \
        cudaError_t e__ = (expr);                                                                     \
        if (e__ != cudaSuccess) {                                                                     \
            char buf__[512];                                                                          \
            std::snprintf(buf__, sizeof buf__, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__, __LINE__); \
            return fail(h, LM_E_CUDA, buf__);                                                         \
        }                                                                                             \
    } while (0)

size_t esize(const lm_solver* h) { return h->precision == LM_F32 ? 4 : 8; }
int64_t dof_of(const lm_solver* h) { return (h->angular ? 6 : 3) * h->N; }

int ensure(lm_solver* h, void** ptr, size_t* cap, size_t bytes)
{
    if (*cap >= bytes && *ptr) return LM_OK;
    if (*ptr) LM_CUDA(h, cudaFree(*ptr));
    *ptr = nullptr;
    *cap = 0;
    LM_CUDA(h, cudaMalloc(ptr, bytes));
    *cap = bytes;
    return LM_OK;
}

// Constants of the pair tensors in the internal length unit: `a` here is a * len_scale; a velocity computed
// from scaled lengths is 1/len_scale times the true one (M_uF ~ 1/r), an angular velocity 1/len_scale^2
// (M_wF ~ 1/r^2; the torques were scaled on packing), hence the two epilogue factors.  All powers of two: exact.
template <typename T> PairConsts<T> make_consts(double eta, double a, double len_scale)
{
    const double pi = 3.14159265358979323846264338327950288;
    PairConsts<T> c;
    const double c4 = 4.0 / (3.0 * a);                 // (1/(6 pi eta a)) / C1: translational self mobility
    const double c8 = 1.0 / (a * a * a);               // (1/(8 pi eta a^3)) / C1: rotational self mobility
    // floor of r^2: r = 0 becomes r = a 2^-40 (fp32) / a 2^-100 (fp64): a relative perturbation of the
    // self term far below the type's epsilon, while 1/r^3 stays finite (1/r^5 may overflow to +inf in
    // fp32; it only feeds the far branch, which the select discards for r < 2a)
    c.tiny = (T)std::max(a * a * std::ldexp(1.0, sizeof(T) == 4 ? -80 : -200), sizeof(T) == 4 ? 4.8e-38 : 1e-300);
    c.four_a2 = (T)(4.0 * a * a);
    c.c2 = (T)(2.0 * a * a / 3.0);
    c.nc3 = (T)(-2.0 * a * a);
    c.c4 = (T)c4;
    c.nc5 = (T)(-c4 * 9.0 / (32.0 * a));
    c.c6 = (T)(c4 * 3.0 / (32.0 * a));
    c.c8 = (T)c8;
    c.k1 = (T)(-c8 * 27.0 / (32.0 * a));
    c.k2 = (T)(c8 * 5.0 / (64.0 * a * a * a));
    c.k3 = (T)(c8 * 9.0 / (32.0 * a));
    c.k4 = (T)(-c8 * 3.0 / (64.0 * a * a * a));
    c.k5 = (T)(1.0 / (2.0 * a * a * a));
    c.k6 = (T)(-3.0 / (16.0 * a * a * a * a));
    c.C1_lin = (T)(len_scale / (8.0 * pi * eta));                  // Oseen prefactor, applied once per target
    c.C1_ang = (T)(len_scale * len_scale / (8.0 * pi * eta));
    c.wa2 = (T)(a * a);
    c.wzz0 = (T)(-8.0 * a * a / 3.0);
    c.wzz1 = (T)(20.0 * a * a);
    return c;
}

template <typename T> std::vector<Variant<T>>& variants(lm_solver* h);
template <> std::vector<Variant<float>>& variants<float>(lm_solver* h) { return h->vf; }
template <> std::vector<Variant<double>>& variants<double>(lm_solver* h) { return h->vd; }

template <typename T> std::vector<SmallVariant<T>>& small_variants(lm_solver* h);
template <> std::vector<SmallVariant<float>>& small_variants<float>(lm_solver* h) { return h->sf; }
template <> std::vector<SmallVariant<double>>& small_variants<double>(lm_solver* h) { return h->sd; }

template <typename T> int init_variants(lm_solver* h)
{
    auto& vs = variants<T>(h);
    vs = build_variants<T>();
    for (auto& v : vs) {
        LM_CUDA(h, cudaFuncSetAttribute((const void*)v.kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, v.smem));
        int nb = 0;
        LM_CUDA(h, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, (const void*)v.kernel, v.block, v.smem));
        v.ctas_per_sm = std::max(nb, 1);
    }
    auto& ss = small_variants<T>(h);
    ss = build_small_variants<T>();
    for (auto& v : ss) LM_CUDA(h, cudaFuncSetAttribute((const void*)v.kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMALL_MAX_SMEM));
    // Can the device co-schedule clusters of this size at all (a MIG slice or a reduced-SM part may not)?  Ask once,
    // for the heaviest shape the chooser may pick; the chooser never exceeds the answer (1 = no clusters: still one launch).
    h->max_cluster = 1;
    for (int S = SM_MAX_CLUSTER; S > 1; S /= 2) {
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(1, S, 1);
        cfg.blockDim = dim3(SM_MAX_WARPS * 32, 1, 1);
        cfg.dynamicSmemBytes = SMALL_MAX_SMEM / 2;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 1;
        attr[0].val.clusterDim.y = S;
        attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        int n = 0;
        if (cudaOccupancyMaxActiveClusters(&n, (const void*)ss[0].kernel, &cfg) == cudaSuccess && n > 0) { h->max_cluster = S; break; }
        (void)cudaGetLastError();
    }
    return LM_OK;
}

// FP-pipe issue cycles one warp spends per source (two targets per lane): the algorithmic lane-operations of
// DESIGN.md sec. 7 x the issue cost of a packed fp32 instruction (2.1 cycles) or of two fp64 ones (2 x 2 cycles).
inline double cycles_per_source(const lm_solver* h, int nrhs)
{
    const double ops = (h->angular ? 16.0 + 32.0 * nrhs : 11.0 + 10.0 * nrhs) + (h->precision == LM_F64 ? 5.0 : 0.0);
    return ops * (h->wall ? 3.4 : 1.0) * (h->precision == LM_F64 ? 4.0 : 2.1);
}

// The shape of the one-launch kernel for this apply, or variant < 0 where the general path (TMA-staged tiles, 2-4
// targets per thread, partials through global memory) is the better one.  A CTA owns 64 targets; its W warps and
// the S CTAs of its cluster split the sources.  Cost model in SM cycles, fitted to phase timings on B200 (clock64
// stamps, N = 256 ... 2048): a lone warp per SM sub-partition is latency-bound (1.3-1.6 x the issue cycles per
// source), warps sharing a sub-partition are issue-bound (x 1.07 fp64, x 1.4 fp32: the packed fp32 body leaves issue
// slots to MUFU / LDS / vote); staging costs ~900 cycles + ~500 per round of 2 elements per thread; the warp sums,
// the push through distributed shared memory, the wait and the final sum ~1300.
template <typename T> SmallPlan choose_small(lm_solver* h, int nrhs)
{
    SmallPlan best;
    if (nrhs < 1 || nrhs > MAX_RHS || h->small_kernel == 0 || h->dist_ranks > 0 || h->acc64) return best;
    auto& slot = h->small_cache[nrhs];
    if (slot.valid && slot.rb == h->row_begin && slot.re == h->row_end && slot.mode == h->small_kernel) return slot.plan;
    const auto& vs = small_variants<T>(h);
    int vi = -1;
    for (int i = 0; i < (int)vs.size(); ++i)
        if (vs[i].nrhs == nrhs && vs[i].ang == h->angular && vs[i].wall == h->wall) vi = i;
    const int64_t rows = std::max<int64_t>(h->row_end - h->row_begin, 0);
    const bool f64 = h->precision == LM_F64;
    const double issue = cycles_per_source(h, nrhs), lone = issue * (f64 ? 1.3 : 1.6), shared = issue * (f64 ? 1.07 : 1.4);
    const bool forced = h->small_kernel > 1;
    // beyond this the general path wins (measured crossovers: fp32 translational N ~ 5000, fp64 ~ 3500;
    // the register-heavy variants -- angular, several right-hand sides: NV = 6 ... 12 accumulated components -- hand over
    // earlier, fp64 more so than fp32)
    const int nv_comp = nrhs * (h->angular ? 6 : 3);
    const double limit = 1.2e9 * (f64 ? 3.0 / nv_comp : std::min(1.0, 6.0 / nv_comp));
    const bool in_range = forced || (double)rows * (double)h->N * issue <= limit;
    if (vi >= 0 && rows > 0 && in_range) {
        const int i_tiles = (int)((rows + SM_TARGETS - 1) / SM_TARGETS);
        double best_cost = 1e300;
        for (int S = 1; S <= h->max_cluster; S *= 2)
            for (int W = 1; W <= SM_MAX_WARPS; W *= 2) {
                if (forced && (S != std::min(h->small_kernel >> 8, h->max_cluster) || W != (h->small_kernel & 255))) continue;
                const int spw = (int)(((h->N + (int64_t)S * W - 1) / ((int64_t)S * W) + 3) / 4 * 4);
                const size_t smem = vs[vi].smem(W, spw);
                if (smem > SMALL_MAX_SMEM) continue;
                // CTAs that fit on one SM at a time (registers, shared memory, threads): more than that run in waves
                int occ = 0;
                if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, (const void*)vs[vi].kernel, W * 32, smem) != cudaSuccess || occ < 1) {
                    (void)cudaGetLastError();
                    continue;
                }
                const double ctas = (double)i_tiles * S, slots = (double)h->sm_count * occ;
                const double full = std::floor(ctas / slots), rem_per_sm = std::ceil((ctas - full * slots) / h->sm_count);
                const double rounds = std::ceil(3.0 * spw / 64.0);
                auto wave = [&](double resident) {            // `resident` CTAs share an SM: their warps share its four sub-partitions
                    return resident > 0 ? spw * std::max(lone, shared * std::ceil(resident * W / 4.0)) + 900.0 + 500.0 * rounds + 1300.0 : 0.0;
                };
                const double cost = full * wave(occ) + wave(rem_per_sm) + 20.0 * (S + W);
                if (cost < best_cost) {
                    best_cost = cost;
                    best.variant = vi;
                    best.i_tiles = i_tiles;
                    best.cluster = S;
                    best.warps = W;
                    best.src_per_warp = spw;
                    best.smem = smem;
                }
            }
    }
    slot.valid = true;
    slot.rb = h->row_begin;
    slot.re = h->row_end;
    slot.mode = h->small_kernel;
    slot.plan = best;
    return best;
}

// Pick the variant and the number of j-splits.  Sources are dealt to the splits in units of SUB, as
// evenly as possible, so the grid can be sized to a whole number of resident sets (148 SMs x
// resident CTAs per SM) whatever N is.  Cost model: CTAs run in waves of `slots`; a CTA costs
// (its sources + a fixed prologue/epilogue) x its targets; CTAs resident on one SM share it.
template <typename T> LaunchPlan choose_plan(lm_solver* h, int nrhs)
{
    if (nrhs >= 0 && nrhs <= MAX_RHS) {
        const auto& slot = h->plan_cache[nrhs];
        if (slot.valid && slot.rb == h->row_begin && slot.re == h->row_end) return slot.plan;
    }
    const auto& vs = variants<T>(h);
    LaunchPlan best;
    double best_cost = 1e300;
    for (int vi = 0; vi < (int)vs.size(); ++vi) {
        const auto& v = vs[vi];
        if (v.nrhs != nrhs || v.ang != h->angular || v.wall != h->wall || v.acc64 != (h->acc64 ? 1 : 0)) continue;
        const int targets = v.block * v.tpt;
        const int64_t rows = std::max<int64_t>(h->row_end - h->row_begin, 0);          // target rows of this rank / call
        const int i_tiles = (int)((rows + targets - 1) / targets);
        const int units = (int)(h->npad / v.sub);
        const int64_t slots = (int64_t)h->sm_count * v.ctas_per_sm;
        const int max_splits = std::min(units, 256);
        const int min_splits = (int)std::min<int64_t>(max_splits, (h->npad + MAX_SOURCES_PER_CTA - 1) / MAX_SOURCES_PER_CTA);
        for (int s = min_splits; s <= max_splits; ++s) {
            if (h->force_splits > 0 && s != std::min(std::max(h->force_splits, min_splits), max_splits)) continue;
            const int64_t src = (int64_t)((units + s - 1) / s) * v.sub;            // sources of the largest split
            const int64_t ctas = (int64_t)i_tiles * s;
            const int64_t full = ctas / slots, rem = ctas % slots;
            const int64_t rem_per_sm = (rem + h->sm_count - 1) / h->sm_count;      // CTAs sharing an SM in the last wave
            // prologue, pipeline fill and epilogue of a CTA ~ 0.03 tile (fitted to plan sweeps on B200)
            const double per_cta = ((double)src + 0.03 * v.tj) * targets / v.efficiency;
            // few resident warps hide less latency: w warps per SM sub-partition cost a factor (1 + 0.3 / w)
            auto wave = [&](int64_t resident) { return resident ? per_cta * resident * (1.0 + 0.3 * 128.0 / ((double)resident * v.block)) : 0.0; };
            double cost = (double)full * wave(v.ctas_per_sm) + wave(rem_per_sm);
            // the SMs do not finish their last CTAs together: ~10 % of the last wave is tail, so several short waves
            // beat one long one (measured: 4 waves 4-5 % faster than 1 at N = 16384 ... 32768, fp32 translational)
            cost += 0.1 * (rem ? wave(rem_per_sm) : wave(v.ctas_per_sm));
            // cost is in pairs evaluated back to back on one SM (~1e4 per microsecond): the reduce pass
            // adds a ~3 us launch plus writing and re-reading s partial vectors
            if (s > 1) cost += (3.0e4 + 0.1 * (double)s * (double)rows) / (h->wall ? 3.4 : 1.0);   // (a wall pair costs ~3.4 free-space pairs)
            if (cost < best_cost) {
                best_cost = cost;
                best.variant = vi;
                best.i_tiles = i_tiles;
                best.j_splits = s;
                best.n_units = units;
            }
        }
    }
    if (nrhs >= 0 && nrhs <= MAX_RHS) {
        auto& slot = h->plan_cache[nrhs];
        slot.valid = true;
        slot.rb = h->row_begin;
        slot.re = h->row_end;
        slot.plan = best;
    }
    return best;
}

cudaEvent_t get_event(lm_solver* h)
{
    if (!h->event_pool.empty()) {
        cudaEvent_t e = h->event_pool.back();
        h->event_pool.pop_back();
        return e;
    }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}

// single wall: the damping factors b (array 4 of the packed positions), and how the packers raise heights
template <typename T> const T* damp_of(const lm_solver* h) { return h->wall ? (const T*)h->pos_soa + (size_t)4 * h->npad : nullptr; }
template <typename T> WallPack<T> wall_pack(const lm_solver* h) { return {h->wall, (T)h->wall_z, (T)(h->a * h->len_scale)}; }
constexpr int POS_ARRAYS = 5;    // x | y | z (raised height with a wall) | height | damping factor  (the last two only with a wall)

int grid_1d(int64_t n) { return (int)std::max<int64_t>(1, (n + VEC_BLOCK - 1) / VEC_BLOCK); }
int grid_red(int64_t n) { return (int)std::min<int64_t>(RED_MAX_BLOCKS, std::max<int64_t>(1, (n + VEC_BLOCK - 1) / VEC_BLOCK)); }


}  // namespace
