// hot_api.cu -- the C ABI of include/hot.h: context, allocations, stage orchestration, exports.
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

#include "hot_internal.h"

long long g_hot_launches = 0;

namespace {

struct Ctx {
    cudaStream_t stream = nullptr;
    Tree t;
    bool built = false;
    int nleaf = 16, ncrit = 256;
    int softening = 0; // 0 Plummer, 1 cubic spline (hot_set_softening)
    int background = 0; // 1: per-cell background subtraction in periodic boxes (hot_set_background)
    uint4 *d_vstack = nullptr, *d_vstage = nullptr, *d_pvlist = nullptr; // virtual cubes of the background-subtracted walk
    int64_t vcap = 4096;        // per-warp capacity of the stack of virtual cubes and of a group's accepted ones; grown fourfold on overflow
    int64_t pv_per_group = 192; // their arena is sized for this many per group; grown fourfold when a walk overflows it
    int last_order = -1, last_tolmode = 0, last_bgmode = 0;
    char err[512] = "";
    // scratch owned across calls
    int* d_flags = nullptr;               // [0] build error bits, [1] hash max probe, [2] forces error bits
    unsigned int* d_counter = nullptr;
    uint4* d_items = nullptr; // work items of the interaction kernel
    unsigned int* d_cls = nullptr; // ... and their per-superblock class counters (launch_plan)
    unsigned long long* d_stat = nullptr; // 4 counters
    uint32_t* d_gstack = nullptr; size_t gstack_bytes = 0; int64_t gstack_cap = 0;
    // device buffers of the build, pooled across hot_build calls: a slot is keyed by the address of
    // the pointer it serves and only ever grows, so a time-stepping caller pays cudaMalloc once
    struct Slot { const void* key; void* p; size_t cap; };
    std::vector<Slot> pool;
    int64_t bytes = 0;
    uint32_t *d_hist = nullptr, *d_counts = nullptr, *d_totals = nullptr;
    int2* d_open = nullptr;
    // interaction lists (hot_forces)
    unsigned long long* d_tops = nullptr;
    double* d_farS = nullptr; // periodic: global moments of the box
    uint32_t *d_pclist = nullptr, *d_pplist = nullptr; uint8_t *d_pcimg = nullptr, *d_ppimg = nullptr;
    uint32_t* d_stage = nullptr; uint8_t* d_stage_img = nullptr; int64_t stage_cap = 0; // per-warp list staging (entries per list)
    unsigned long long arena_pc = 0, arena_pp = 0; // entries the list arena holds
    unsigned long long used_pc = 0, used_pp = 0;   // entries the last hot_forces wrote (sizes the next arena)
    int64_t used_groups = 0, last_n = 0; int last_periodic = -1;
    size_t arena_cap_bytes = 0;                     // 0 = as much as fits; else a cap (hot_set_list_arena)
    std::vector<cudaEvent_t> evx;
    bool lists_valid = false;
    hot_stats_t st{};
    cudaEvent_t ev[9] = {};
    bool ev_ready = false;
    int64_t list_g0 = 0, list_g1 = 0; // groups whose lists the arena holds after the last hot_forces
    // device staging of hot_step_host
    int64_t h_n = 0;
    float *hd_pos = nullptr, *hd_mass = nullptr, *hd_acc = nullptr, *hd_pot = nullptr;
};
Ctx g;

int fail(int code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g.err, sizeof(g.err), fmt, ap);
    va_end(ap);
    return code;
}
#define CUDA_TRY(expr)                                                                                   \
    do {                                                                                                 \
        cudaError_t e_ = (expr);                                                                         \
        if (e_ != cudaSuccess) {                                                                         \
            int code_ = e_ == cudaErrorMemoryAllocation ? HOT_ENOMEM : HOT_ECUDA;                        \
            cudaGetLastError();                                                                          \
            return fail(code_, "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
        }                                                                                                \
    } while (0)

template <typename T> cudaError_t tree_alloc(T** p, size_t count) {
    size_t bytes = count * sizeof(T);
    if (bytes == 0) bytes = sizeof(T);
    Ctx::Slot* s = nullptr;
    for (auto& q : g.pool) if (q.key == (const void*)p) { s = &q; break; }
    if (!s) { g.pool.push_back({(const void*)p, nullptr, 0}); s = &g.pool.back(); }
    if (s->cap < bytes) {
        if (s->p) { cudaFree(s->p); g.bytes -= (int64_t)s->cap; s->p = nullptr; s->cap = 0; }
        size_t want = bytes + bytes / 8; // headroom: cell counts drift from step to step
        cudaError_t e = cudaMalloc(&s->p, want);
        if (e != cudaSuccess) { cudaGetLastError(); want = bytes; e = cudaMalloc(&s->p, want); }
        if (e != cudaSuccess) { s->p = nullptr; return e; }
        s->cap = want;
        g.bytes += (int64_t)want;
    }
    *p = static_cast<T*>(s->p);
    return cudaSuccess;
}
void release_pool() {
    for (auto& q : g.pool) cudaFree(q.p);
    g.pool.clear();
    g.bytes = 0;
}
void drop_build() { // forgets the build; its buffers stay pooled for the next one
    int nleaf = g.t.nleaf, ncrit = g.t.ncrit;
    g.t = Tree();
    g.t.nleaf = nleaf; g.t.ncrit = ncrit;
    g.built = false;
    g.last_order = -1;
    g.lists_valid = false;
}
int ensure_scratch() {
    if (!g.d_flags) {
        CUDA_TRY(cudaMalloc(&g.d_flags, 4 * sizeof(int)));
        CUDA_TRY(cudaMalloc(&g.d_counter, 2 * sizeof(unsigned int))); // walk and interaction schedulers
        CUDA_TRY(cudaMalloc(&g.d_stat, 6 * sizeof(unsigned long long)));
    }
    if (!g.ev_ready) {
        for (auto& e : g.ev) CUDA_TRY(cudaEventCreate(&e));
        g.ev_ready = true;
    }
    return HOT_OK;
}
// MAC thresholds (R-7): the criterion is  (double)(s*s) < theta2 * (double)d2  with s = 2^(21-l)
// and d2 an integer < 2^53.  fl(theta2 * d2) is non-decreasing in d2, so for every level there is one
// smallest integer T[l] with the criterion true for exactly the d2 >= T[l]; it is found by bisection
// with that same IEEE double multiply and compare, and the kernel tests d2 >= T[l] in integers.
void mac_table(double theta2, unsigned long long* T) {
    for (int l = 0; l < HOT_NLEVELS; ++l) {
        const double s2 = std::ldexp(1.0, 2 * (HOT_MAXLEVEL - l));
        auto ok = [&](unsigned long long d2) { volatile double p = theta2 * (double)d2; return s2 < p; };
        unsigned long long lo = 0, hi = 1ull << 53; // lo fails (0 is never accepted), hi is tested first
        if (!ok(hi)) { T[l] = ~0ull; continue; }
        while (hi - lo > 1) { const unsigned long long mid = lo + (hi - lo) / 2; if (ok(mid)) hi = mid; else lo = mid; }
        T[l] = hi;
    }
}
float ms_between(cudaEvent_t a, cudaEvent_t b) {
    float ms = 0;
    if (cudaEventElapsedTime(&ms, a, b) != cudaSuccess) { cudaGetLastError(); ms = 0; }
    return ms;
}

} // namespace

extern "C" {

const char* hot_last_error(void) { return g.err; }

int hot_set_stream(void* s) {
    g.stream = static_cast<cudaStream_t>(s);
    return HOT_OK;
}

int hot_measure_fp32(double* tflops_scalar, double* tflops_packed) {
    if (!tflops_scalar || !tflops_packed) return fail(HOT_EINVAL, "hot_measure_fp32: NULL output");
    CUDA_TRY(measure_fp32(tflops_scalar, tflops_packed, g.stream));
    return HOT_OK;
}

int hot_measure_fp32_operands(double* tflops3) {
    if (!tflops3) return fail(HOT_EINVAL, "hot_measure_fp32_operands: NULL output");
    CUDA_TRY(measure_fp32_operands(tflops3, g.stream));
    return HOT_OK;
}

int hot_far_coefficients(double* coef165) {
    if (!coef165) return fail(HOT_EINVAL, "hot_far_coefficients: NULL output");
    far_coefficients(coef165);
    return HOT_OK;
}

int hot_set_list_arena(int64_t max_bytes) {
    if (max_bytes < 0) return fail(HOT_EINVAL, "hot_set_list_arena: max_bytes must be >= 0");
    g.arena_cap_bytes = (size_t)max_bytes;
    return HOT_OK;
}

int hot_set_params(int nleaf, int ncrit) {
    if (nleaf < 1 || nleaf > HOT_MAX_NLEAF || ncrit < nleaf || ncrit > HOT_MAX_NCRIT)
        return fail(HOT_EINVAL, "hot_set_params: need 1 <= nleaf <= %d, nleaf <= ncrit <= %d", HOT_MAX_NLEAF, HOT_MAX_NCRIT);
    g.nleaf = nleaf; g.ncrit = ncrit;
    return HOT_OK;
}

int hot_set_softening(int kind) {
    if (kind != 0 && kind != 1) return fail(HOT_EINVAL, "hot_set_softening: kind must be 0 (Plummer) or 1 (cubic spline)");
    g.softening = kind;
    return HOT_OK;
}

int hot_set_background(int on) {
    if (on != 0 && on != 1) return fail(HOT_EINVAL, "hot_set_background: 0 or 1");
    g.background = on;
    return HOT_OK;
}

int hot_kick_drift(float* pos, float* vel, const float* acc, int64_t n, float dt_kick, float dt_drift, hot_box box, int periodic) {
    if (!pos || !vel || !acc) return fail(HOT_EINVAL, "hot_kick_drift: NULL argument");
    if (n < 1) return fail(HOT_EINVAL, "hot_kick_drift: n must be >= 1");
    if (periodic && !(box.size > 0.0f)) return fail(HOT_EINVAL, "hot_kick_drift: box.size must be positive");
    CUDA_TRY(launch_kick_drift(pos, vel, acc, n, dt_kick, dt_drift, box.lo[0], box.lo[1], box.lo[2], box.size, periodic ? 1 : 0, g.stream));
    return HOT_OK;
}

void hot_free(void) {
    drop_build();
    release_pool();
    cudaFree(g.d_flags); cudaFree(g.d_counter); cudaFree(g.d_stat); cudaFree(g.d_gstack);
    g.d_flags = nullptr; g.d_counter = nullptr; g.d_stat = nullptr; g.d_gstack = nullptr; g.gstack_bytes = 0;
    if (g.ev_ready) { for (auto& e : g.ev) cudaEventDestroy(e); g.ev_ready = false; }
    for (auto& e : g.evx) cudaEventDestroy(e);
    g.evx.clear();
    g.arena_pc = g.arena_pp = 0; g.used_pc = g.used_pp = 0; g.used_groups = 0; g.stage_cap = 0;
    cudaFree(g.hd_pos); cudaFree(g.hd_mass); cudaFree(g.hd_acc); cudaFree(g.hd_pot);
    g.hd_pos = g.hd_mass = g.hd_acc = g.hd_pot = nullptr; g.h_n = 0;
    cudaGetLastError();
    g.st = hot_stats_t{};
}

int hot_build(const float* pos, const float* mass, int64_t n, hot_box box, int periodic) {
    if (!pos || !mass) return fail(HOT_EINVAL, "hot_build: NULL pos or mass");
    if (n < 1 || n > ((int64_t)1 << 27)) return fail(HOT_EINVAL, "hot_build: n = %lld outside [1, 2^27]", (long long)n);
    if (!(box.size > 0.0f) || !(box.size < 3.0e38f)) return fail(HOT_EINVAL, "hot_build: box.size must be positive and finite");
    if (periodic != 0 && periodic != 1) return fail(HOT_EINVAL, "hot_build: periodic must be 0 or 1");
    int rc = ensure_scratch();
    if (rc) return rc;
    drop_build();
    g_hot_launches = 0;
    if (g.last_n != n || g.last_periodic != periodic) { g.used_pc = g.used_pp = 0; g.used_groups = 0; } // another problem: forget its list sizes
    g.last_n = n; g.last_periodic = periodic;
    Tree& t = g.t;
    t.n = n; t.periodic = periodic; t.nleaf = g.nleaf; t.ncrit = g.ncrit; t.box = box;
    for (int k = 0; k < 3; ++k) t.lo[k] = (double)box.lo[k];
    t.size = (double)box.size;
    cudaStream_t st = g.stream;
    const float inv = 1.0f / box.size; // one IEEE fp32 division on the host: part of the key's definition

    struct Guard { bool ok = false; ~Guard() { if (!ok) drop_build(); } } guard;

    uint32_t *&d_hist = g.d_hist, *&d_counts = g.d_counts, *&d_totals = g.d_totals;
    const int64_t nblk = tree_num_blocks(n);
    const int rows = HOT_NLEVELS + 2;
    CUDA_TRY(tree_alloc(&t.key[0], (size_t)n));
    CUDA_TRY(tree_alloc(&t.key[1], (size_t)n));
    CUDA_TRY(tree_alloc(&t.idx[0], (size_t)n));
    CUDA_TRY(tree_alloc(&t.idx[1], (size_t)n));
    CUDA_TRY(tree_alloc(&t.body, (size_t)n));
    CUDA_TRY(tree_alloc(&t.bin, (size_t)n));
    CUDA_TRY(tree_alloc(&t.plev, (size_t)n));
    CUDA_TRY(tree_alloc(&d_hist, sort_hist_elems(n)));
    CUDA_TRY(tree_alloc(&d_counts, (size_t)rows * (size_t)nblk));
    CUDA_TRY(tree_alloc(&g.d_open, (size_t)HOT_NLEVELS * (size_t)nblk));
    CUDA_TRY(tree_alloc(&d_totals, (size_t)rows));
    CUDA_TRY(cudaMemsetAsync(g.d_flags, 0, 4 * sizeof(int), st));

    CUDA_TRY(cudaEventRecord(g.ev[0], st));
    CUDA_TRY(launch_keygen(pos, mass, n, box.lo[0], box.lo[1], box.lo[2], inv, t.key[0], t.bin, d_hist, g.d_flags, st));
    CUDA_TRY(cudaEventRecord(g.ev[1], st));
    CUDA_TRY(launch_radix_sort(t.key, t.idx, n, d_hist, st));
    CUDA_TRY(cudaEventRecord(g.ev[2], st));
    CUDA_TRY(launch_gather(t.bin, t.idx[0], n, t.body, st));
    CUDA_TRY(cudaEventRecord(g.ev[3], st));
    CUDA_TRY(launch_tree_levels(t.key[0], n, t.nleaf, t.ncrit, t.plev, d_counts, st));
    CUDA_TRY(launch_tree_scan(d_counts, nblk, d_totals, st));
    uint32_t totals[HOT_NLEVELS + 2];
    int flags[4];
    CUDA_TRY(cudaMemcpyAsync(totals, d_totals, sizeof(totals), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(flags, g.d_flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (flags[0] & 1) return fail(HOT_ERANGE, "hot_build: a particle lies outside [lo, lo+size)^3");
    t.level_base[0] = 0;
    t.max_level = 0;
    for (int l = 0; l < HOT_NLEVELS; ++l) {
        t.level_base[l + 1] = t.level_base[l] + (int64_t)totals[l];
        if (totals[l]) t.max_level = l;
    }
    t.ncells = t.level_base[HOT_NLEVELS];
    t.ngroups = (int64_t)totals[HOT_NLEVELS];
    t.nleaves = (int64_t)totals[HOT_NLEVELS + 1];
    if (t.ncells >= ((int64_t)1 << 28)) return fail(HOT_EINTERNAL, "hot_build: %lld cells exceed the 28-bit cell index of the walk", (long long)t.ncells);
    t.hcap = 64;
    while (t.hcap < 2 * t.ncells) t.hcap <<= 1;
    CUDA_TRY(tree_alloc(&t.ckey, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.cfirst, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.ccount, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.cmask, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.cchild, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.cparent, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.wcell, (size_t)t.ncells));
    CUDA_TRY(tree_alloc(&t.group, (size_t)t.ngroups));
    CUDA_TRY(tree_alloc(&t.leafcell, (size_t)t.nleaves));
    CUDA_TRY(tree_alloc(&t.glpc, (size_t)t.ngroups));
    CUDA_TRY(tree_alloc(&t.glpp, (size_t)t.ngroups));
    CUDA_TRY(tree_alloc(&t.hval, (size_t)t.hcap));
    CUDA_TRY(cudaMemsetAsync(t.hval, 0xff, sizeof(int32_t) * (size_t)t.hcap, st)); // -1: free slot
    CUDA_TRY(cudaMemsetAsync(t.glpc, 0, sizeof(uint32_t) * (size_t)t.ngroups, st));
    CUDA_TRY(cudaMemsetAsync(t.glpp, 0, sizeof(uint32_t) * (size_t)t.ngroups, st));
    TreeEmitArgs ea;
    ea.skey = t.key[0]; ea.plev = t.plev; ea.counts = d_counts; ea.n = n; ea.nblk = nblk;
    for (int l = 0; l <= HOT_NLEVELS; ++l) ea.level_base[l] = t.level_base[l];
    ea.ckey = t.ckey; ea.cfirst = t.cfirst; ea.ccount = t.ccount; ea.cchild = t.cchild; ea.cparent = t.cparent;
    ea.group = t.group; ea.leafcell = t.leafcell; ea.open = g.d_open;
    CUDA_TRY(launch_tree_emit(ea, st));
    CUDA_TRY(launch_tree_link(t.ckey, t.ncells, t.hval, t.hcap - 1, g.d_flags + 1, st));
    CUDA_TRY(launch_tree_finalize(t.ckey, t.cfirst, t.ccount, t.cmask, t.cchild, t.wcell, t.ncells, g.d_flags, st));
    CUDA_TRY(cudaEventRecord(g.ev[4], st));
    CUDA_TRY(cudaMemcpyAsync(flags, g.d_flags, sizeof(flags), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (flags[0] & 2) return fail(HOT_ERANGE, "hot_build: 2^27 or more coincident bodies in one finest-level cell");
    t.hash_max_probe = flags[1];

    hot_stats_t& s = g.st;
    s = hot_stats_t{};
    s.n = n; s.n_cells = t.ncells; s.n_leaves = t.nleaves; s.n_groups = t.ngroups; s.max_level = t.max_level;
    s.nleaf = t.nleaf; s.ncrit = t.ncrit; s.periodic = periodic; s.hash_capacity = t.hcap; s.hash_max_probe = t.hash_max_probe;
    s.order = -1;
    s.ms_keygen = ms_between(g.ev[0], g.ev[1]);
    s.ms_sort = ms_between(g.ev[1], g.ev[2]);
    s.ms_gather = ms_between(g.ev[2], g.ev[3]);
    s.ms_tree = ms_between(g.ev[3], g.ev[4]);
    s.ms_build_total = ms_between(g.ev[0], g.ev[4]);
    s.bytes_allocated = g.bytes;
    s.launches_build = g_hot_launches;
    guard.ok = true;
    g.built = true;
    return HOT_OK;
}

} // extern "C"
namespace {
// hot_forces (tolmode 0: opening angle theta, one expansion order) and hot_forces_tol (tolmode 1: error-bound criterion
// with the order chosen per interaction, R-16) share everything but the criterion and the evaluation launches
int forces_impl(const int tolmode, const double theta, const double tol, const double eps, int order, float* acc, float* pot) {
    Tree& t = g.t;
    cudaStream_t st = g.stream;
    g_hot_launches = 0;
    CUDA_TRY(cudaEventRecord(g.ev[5], st));
    // S6: moments, cached per build at the highest order asked so far
    if (t.mom_order < order) {
        if (!t.cellA) CUDA_TRY(tree_alloc(&t.cellA, (size_t)t.ncells));
        if (t.periodic && !t.cellM0d) CUDA_TRY(tree_alloc(&t.cellM0d, (size_t)t.ncells));
        if (order >= 2 && !t.cellM2) { CUDA_TRY(tree_alloc(&t.cellM2, (size_t)t.ncells)); CUDA_TRY(tree_alloc(&t.cellE2, (size_t)t.ncells)); }
        if (order >= 4 && !t.cellM34) { CUDA_TRY(tree_alloc(&t.cellM34, (size_t)t.ncells)); CUDA_TRY(tree_alloc(&t.cellMac, (size_t)t.ncells)); }
        if (order >= 6) { // f-3: raw moments of degree 5 .. order and their trace record (gen_hi_orders.py), in units of the cell side
            CUDA_TRY(tree_alloc(&t.cellHiRaw, (size_t)t.ncells * (size_t)hi_raw_floats(order)));
            CUDA_TRY(tree_alloc(&t.cellHiT, (size_t)t.ncells * (size_t)hi_record_floats(order)));
            t.hi_order = order;
        }
        CUDA_TRY(launch_moments(t, order, st));
        t.mom_order = order;
    }
    CUDA_TRY(cudaEventRecord(g.ev[6], st));
    int rc = HOT_OK;
    // P2/P3: what the 125 explicit boxes leave of the periodic sum, and the background (hot_periodic.cu);
    // per body in fp64, added by the interaction kernel before its one rounding to fp32
    if (t.periodic) {
        if (!t.far_ready) { // global moments of the box and the per-body far field: once per build
            CUDA_TRY(tree_alloc(&g.d_farS, 165));
            CUDA_TRY(tree_alloc(&t.far, 4 * (size_t)t.n));
            CUDA_TRY(tree_alloc(&t.farc, 4 * (size_t)t.n));
            CUDA_TRY(launch_far_moments(t, g.d_farS, st));
            double S[165];
            CUDA_TRY(cudaMemcpyAsync(S, g.d_farS, sizeof(S), cudaMemcpyDeviceToHost, st));
            CUDA_TRY(cudaStreamSynchronize(st));
            far_sink_polynomial(S, t.farD);
            t.total_mass = S[0];
            CUDA_TRY(launch_far_eval(t, t.farD, t.far, st)); // depends on the bodies only: kept for every hot_forces on this build
            t.far_ready = true;
        }
    }
    const int bgmode = t.periodic && g.background && !tolmode && order <= 4; // f-1 (R-18)
    const double rhobar = t.total_mass / (t.size * t.size * t.size);
    if (bgmode && t.bg_order != order) { // moments about the cell centres minus the uniform cube's, through the same order
        CUDA_TRY(tree_alloc(&t.bgA, (size_t)t.ncells));
        if (order >= 2) CUDA_TRY(tree_alloc(&t.bgE2, (size_t)t.ncells));
        if (order >= 4) CUDA_TRY(tree_alloc(&t.bgM34, (size_t)t.ncells));
        CUDA_TRY(launch_bg_moments(t, order, rhobar, st));
        t.bg_order = order;
    }
    CUDA_TRY(cudaEventRecord(g.ev[8], st));
    // S7: the walk writes every group's lists into the arena; S8/S9/S10 evaluate them.  The arena is
    // sized from the previous call (first call: a guess); if it is too small the walk reports the
    // first group that did not fit, the groups before it are evaluated and the walk goes on from there.
    const int nwarps = walk_grid_warps();
    const int64_t gcap = 4096; // spill arena entries per warp
    size_t need = (size_t)nwarps * (size_t)gcap * sizeof(uint32_t) * (t.periodic ? 2 : 1);
    if (need > g.gstack_bytes) {
        cudaFree(g.d_gstack); g.d_gstack = nullptr; g.gstack_bytes = 0;
        CUDA_TRY(cudaMalloc(&g.d_gstack, need));
        g.gstack_bytes = need;
    }
    const int64_t ng = t.ngroups;
    CUDA_TRY(tree_alloc(&t.glvis, (size_t)ng));
    CUDA_TRY(tree_alloc(&t.pcoff, (size_t)ng));
    CUDA_TRY(tree_alloc(&t.ppoff, (size_t)ng));
    CUDA_TRY(tree_alloc(&g.d_tops, 3));
    const size_t esz = t.periodic ? 5 : 4; // bytes per list entry: u32 (+ u8 image id)
    if (g.stage_cap < 1024) g.stage_cap = 16384;
    // a group's cell list cannot hold more than every cell of every image, nor its run list more than one run per leaf and
    // per 32 bodies: small problems get a small staging area (it is nwarps x 2 x stage_cap words: 0.8 GB at 16384)
    int64_t stage_use = g.stage_cap;
    {
        const int64_t most = (t.periodic ? 125 : 1) * (t.ncells + t.n / 32 + 1);
        if (most < stage_use) stage_use = most < 1024 ? 1024 : ((most + 1023) / 1024) * 1024;
    }
    // arena capacity in entries: what the last call needed plus 12%, else a first guess
    unsigned long long cappc = g.used_pc ? g.used_pc + g.used_pc / 8 + 4096 : (unsigned long long)ng * (t.periodic ? 6000 : 2800) + 65536;
    unsigned long long cappp = g.used_pp ? g.used_pp + g.used_pp / 8 + 4096 : (unsigned long long)ng * (t.periodic ? 3000 : 1400) + 65536;
    if (cappc < g.arena_pc) cappc = g.arena_pc; // never shrink what the pool already holds
    if (cappp < g.arena_pp) cappp = g.arena_pp;
    auto clamp_arena = [&]() -> int {
        size_t fre = 0, tot = 0;
        CUDA_TRY(cudaMemGetInfo(&fre, &tot));
        double have = 0.7 * (double)fre + (double)(g.arena_pc + g.arena_pp) * (double)esz; // what the pool holds counts as available
        if (g.arena_cap_bytes > 0 && (double)g.arena_cap_bytes < have) have = (double)g.arena_cap_bytes; // hot_set_list_arena
        const double want = (double)(cappc + cappp) * (double)esz;
        if (want > have) { const double f = have / want; cappc = (unsigned long long)(cappc * f) + 1; cappp = (unsigned long long)(cappp * f) + 1; }
        return HOT_OK;
    };
    if (cappc > g.arena_pc || cappp > g.arena_pp || g.arena_cap_bytes > 0) { rc = clamp_arena(); if (rc) return rc; }
    auto alloc_lists = [&]() -> int {
        CUDA_TRY(tree_alloc(&g.d_pclist, (size_t)cappc));
        CUDA_TRY(tree_alloc(&g.d_pplist, (size_t)cappp));
        if (t.periodic) { CUDA_TRY(tree_alloc(&g.d_pcimg, (size_t)cappc)); CUDA_TRY(tree_alloc(&g.d_ppimg, (size_t)cappp)); }
        g.arena_pc = cappc; g.arena_pp = cappp;
        return HOT_OK;
    };
    auto alloc_stage = [&]() -> int {
        CUDA_TRY(tree_alloc(&g.d_stage, (size_t)nwarps * 2 * (size_t)stage_use));
        if (t.periodic) CUDA_TRY(tree_alloc(&g.d_stage_img, (size_t)nwarps * 2 * (size_t)stage_use));
        return HOT_OK;
    };
    rc = alloc_lists(); if (rc) return rc;
    rc = alloc_stage(); if (rc) return rc;
    CUDA_TRY(cudaMemsetAsync(g.d_stat, 0, 6 * sizeof(unsigned long long), st));
    CUDA_TRY(cudaMemsetAsync(g.d_flags + 2, 0, sizeof(int), st));
    WalkArgs wa{};
    wa.wcell = t.wcell; wa.group = t.group; wa.g1 = ng;
    mac_table(theta * theta, wa.mac_t); // theta^2 formed once on the host in double (R-7)
    const double hreal = g.softening == 1 ? 2.8 * eps : 0.0; // spline softening: support radius of a body (R-17)
    if (g.softening == 1) { // an accepted cell lies beyond h: d2 > (h / grid spacing)^2, folded into the integer thresholds
        const double hg = hreal * 2097152.0 / t.size, hgrid2 = hg * hg;
        const unsigned long long need = hgrid2 < 9.0e18 ? (unsigned long long)std::floor(hgrid2) + 1ull : ~0ull;
        for (int l = 0; l < HOT_NLEVELS; ++l) if (wa.mac_t[l] < need) wa.mac_t[l] = need;
    }
    wa.hreal = hreal;
    wa.tolmode = tolmode; wa.tol = tol; wa.size = t.size; wa.cellA = t.cellA; wa.cellMac = t.cellMac;
    for (int k = 0; k < 3; ++k) wa.lo[k] = t.lo[k];
    if (tolmode || bgmode) { CUDA_TRY(tree_alloc(&t.glpc0, (size_t)ng)); CUDA_TRY(tree_alloc(&t.glpc2, (size_t)ng)); }
    wa.bgmode = bgmode; wa.cmask = t.cmask;
    int64_t vstack_cap = g.vcap, vstage_cap = g.vcap;
    unsigned long long cappv = 0;
    if (bgmode) {
        CUDA_TRY(tree_alloc(&g.d_vstack, (size_t)nwarps * (size_t)vstack_cap));
        CUDA_TRY(tree_alloc(&g.d_vstage, (size_t)nwarps * (size_t)vstage_cap));
        cappv = (unsigned long long)ng * (unsigned long long)g.pv_per_group + 65536ull;
        CUDA_TRY(tree_alloc(&g.d_pvlist, (size_t)cappv));
        CUDA_TRY(tree_alloc(&t.glpv, (size_t)ng));
        CUDA_TRY(tree_alloc(&t.gpvoff, (size_t)ng));
    }
    wa.vstack = g.d_vstack; wa.vstack_cap = vstack_cap; wa.vstage = g.d_vstage; wa.vstage_cap = vstage_cap;
    wa.pvlist = g.d_pvlist; wa.cappv = cappv; wa.lpv = t.glpv; wa.pvoff = t.gpvoff;
    wa.lpc0 = t.glpc0; wa.lpc2 = t.glpc2;
    wa.periodic = t.periodic; wa.lpc = t.glpc; wa.lpp = t.glpp; wa.lvis = t.glvis; wa.pcoff = t.pcoff; wa.ppoff = t.ppoff;
    wa.tops = g.d_tops; wa.first_fail = g.d_flags + 3;
    wa.counter = g.d_counter; wa.stat = g.d_stat; wa.gstack = g.d_gstack; wa.gstack_cap = gcap; wa.errflag = g.d_flags + 2;
    ForceArgs a{};
    a.wcell = t.wcell; a.cellA = t.cellA; a.cellE2 = t.cellE2; a.cellM34 = t.cellM34;
    a.body = t.body; a.perm = t.idx[0]; a.group = t.group;
    a.pcoff = t.pcoff; a.ppoff = t.ppoff; a.lpc = t.glpc; a.lpp = t.glpp;
    a.eps2 = (float)(eps * eps); a.order = order > 4 ? 4 : order; a.periodic = t.periodic; // orders 6, 8: the kernels of hot_forces.cu through 4, hot_hi.cu adds the rest
    a.spline = g.softening == 1; a.hinv = hreal > 0.0 ? (float)(1.0 / hreal) : INFINITY;
    for (int k = 0; k < 3; ++k) a.lo[k] = t.lo[k];
    a.size = t.size;
    a.far = t.periodic ? t.far : nullptr;
    a.seg = -1; a.lpc0 = t.glpc0; a.lpc2 = t.glpc2; a.do_pp = 1; a.accumulate = 0;
    a.acc = acc; a.pot = pot; a.counter = g.d_counter + 1;
    a.sb_shift = 16; // 2^16 sink groups per superblock of the work-item order (hot_forces.cu; 2^13 ... whole set measured equal, smaller slower)
    CUDA_TRY(tree_alloc(&g.d_cls, plan_cls_elems(ng, a.sb_shift)));
    a.cls = g.d_cls;
    CUDA_TRY(tree_alloc(&g.d_items, (size_t)(HOT_MAX_NCRIT / 64 + 2) * (size_t)ng)); // passes per group: full ones of >= 64 sinks, one split in two
    a.items = g.d_items;
    // groups per round: all of them unless the arena is known (or found) to be too small.  The warps
    // take arena slices in completion order, so in an overfull round the FIRST group may be among
    // those that fail: then the round is repeated with a quarter of the groups.
    int64_t budget = ng;
    if (g.used_pc + g.used_pp > 0 && g.used_groups > 0) {
        const double per_group = (double)(g.used_pc + g.used_pp) / (double)g.used_groups;
        const double fit = 0.85 * (double)(cappc + cappp) / (per_group > 1.0 ? per_group : 1.0);
        if (fit < 0.8 * (double)ng) budget = fit < 1.0 ? 1 : (int64_t)fit; // clearly too small (a capped arena): plan the rounds
    }
    int64_t g0 = 0;
    size_t nrounds = 0;
    unsigned long long usedpc = 0, usedpp = 0;
    float ms_walk = 0, ms_eval = 0, ms_coarse = 0;
    if (g.evx.size() < 5) { while (g.evx.size() < 5) { cudaEvent_t e; CUDA_TRY(cudaEventCreate(&e)); g.evx.push_back(e); } }
    while (g0 < ng) {
        const int ff0 = INT_MAX;
        CUDA_TRY(cudaMemsetAsync(g.d_counter, 0, 2 * sizeof(unsigned int), st));
        CUDA_TRY(cudaMemsetAsync(g.d_tops, 0, 3 * sizeof(unsigned long long), st));
        CUDA_TRY(cudaMemcpyAsync(g.d_flags + 3, &ff0, sizeof(int), cudaMemcpyHostToDevice, st));
        wa.g0 = g0; wa.g1 = g0 + budget < ng ? g0 + budget : ng;
        wa.pclist = g.d_pclist; wa.pplist = g.d_pplist; wa.pcimg = g.d_pcimg; wa.ppimg = g.d_ppimg; wa.cappc = cappc; wa.cappp = cappp;
        wa.stage = g.d_stage; wa.stage_img = g.d_stage_img; wa.stage_cap = stage_use;
        CUDA_TRY(cudaEventRecord(g.evx[0], st));
        CUDA_TRY(launch_walk(wa, st));
        CUDA_TRY(cudaEventRecord(g.evx[1], st));
        int fl[2] = {0, 0}; // errflag, first_fail
        unsigned long long tops[2] = {0, 0};
        CUDA_TRY(cudaMemcpyAsync(fl, g.d_flags + 2, 2 * sizeof(int), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaMemcpyAsync(tops, g.d_tops, sizeof(tops), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        ms_walk += ms_between(g.evx[0], g.evx[1]);
        if (fl[0] & 4) return fail(HOT_EINTERNAL, "hot_forces: traversal scratch exhausted");
        if (fl[0] & 16) { // a group's virtual cubes outgrew the per-warp scratch (sparse sets: much empty space to tile): enlarge it, walk again
            if (g.vcap >= ((int64_t)1 << 20)) return fail(HOT_EINTERNAL, "hot_forces: virtual-cube scratch of the background-subtracted walk exhausted");
            g.vcap *= 4; vstack_cap = vstage_cap = g.vcap;
            CUDA_TRY(tree_alloc(&g.d_vstack, (size_t)nwarps * (size_t)vstack_cap));
            CUDA_TRY(tree_alloc(&g.d_vstage, (size_t)nwarps * (size_t)vstage_cap));
            wa.vstack = g.d_vstack; wa.vstack_cap = vstack_cap; wa.vstage = g.d_vstage; wa.vstage_cap = vstage_cap;
            CUDA_TRY(cudaMemsetAsync(g.d_flags + 2, 0, sizeof(int), st));
            continue;
        }
        if (fl[0] & 32) { // the accepted virtual cubes outgrew their arena: enlarge it and walk this range again
            if (g.pv_per_group >= (1 << 16)) return fail(HOT_ENOMEM, "hot_forces: the virtual-cube list of the background-subtracted walk does not fit its arena");
            g.pv_per_group *= 4;
            cappv = (unsigned long long)ng * (unsigned long long)g.pv_per_group + 65536ull;
            CUDA_TRY(tree_alloc(&g.d_pvlist, (size_t)cappv));
            wa.pvlist = g.d_pvlist; wa.cappv = cappv;
            CUDA_TRY(cudaMemsetAsync(g.d_flags + 2, 0, sizeof(int), st));
            continue;
        }
        if (fl[0] & 8) { // a group's lists outgrew the per-warp staging area: enlarge it and walk this range again
            if (g.stage_cap >= ((int64_t)1 << 26)) return fail(HOT_ENOMEM, "hot_forces: one sink group's interaction list exceeds 2^26 entries");
            g.stage_cap = stage_use * 4; stage_use = g.stage_cap;
            rc = alloc_stage(); if (rc) return rc;
            CUDA_TRY(cudaMemsetAsync(g.d_flags + 2, 0, sizeof(int), st));
            continue;
        }
        const int64_t F = fl[1] < wa.g1 ? (int64_t)fl[1] : wa.g1;
        if (F == g0 && wa.g1 - g0 > 1) { budget = (wa.g1 - g0) / 4 > 1 ? (wa.g1 - g0) / 4 : 1; continue; }
        if (F == g0) { // one group alone does not fit: enlarge the arena if memory allows
            const unsigned long long oldpc = cappc, oldpp = cappp;
            cappc *= 2; cappp *= 2;
            rc = clamp_arena(); if (rc) return rc;
            if (cappc <= oldpc + oldpc / 16 && cappp <= oldpp + oldpp / 16)
                return fail(HOT_ENOMEM, "hot_forces: the interaction lists of one sink group do not fit the list arena (%llu + %llu entries)", oldpc, oldpp);
            if (cappc < oldpc) cappc = oldpc;
            if (cappp < oldpp) cappp = oldpp;
            rc = alloc_lists(); if (rc) return rc;
            continue;
        }
        // tops also counts what groups that did not fit asked for: no more than the arena was really written
        usedpc += tops[0] < cappc ? tops[0] : cappc; usedpp += tops[1] < cappp ? tops[1] : cappp;
        a.g0 = g0; a.g1 = F;
        a.nsb = (unsigned int)((F - g0 + ((int64_t)1 << a.sb_shift) - 1) >> a.sb_shift);
        a.pclist = g.d_pclist; a.pplist = g.d_pplist; a.pcimg = g.d_pcimg; a.ppimg = g.d_ppimg;
        CUDA_TRY(launch_plan(a, st));
        if (bgmode) { // hot_bg.cu: far field + background added back + virtual cubes -> farc (fp64); then the flagged cells about
                      // their centres through the blocked kernel, added to farc; the launch below takes the plain near field
            CUDA_TRY(cudaEventRecord(g.evx[4], st));
            a.lpc0 = t.glpc0; a.lpc2 = t.glpc2;
            CUDA_TRY(launch_forces_bg(a, t, t.far, t.farc, g.d_pvlist, t.glpv, t.gpvoff, rhobar, 0, st));
            ForceArgs b = a;
            b.seg = 1; b.do_pp = 0; b.bgv = 1; b.bgA = t.bgA; b.bgE2 = t.bgE2; b.bgM34 = t.bgM34; b.out_farc = t.farc; b.far = nullptr;
            if (g.softening == 1) b.eps2 = 0.0f; // spline: accepted cells are Newtonian
            CUDA_TRY(launch_forces(b, st));
            CUDA_TRY(cudaMemsetAsync(g.d_counter + 1, 0, sizeof(unsigned int), st)); // the work-item scheduler starts over
            a.far = t.farc; a.seg = 0; // the plain cells (inside the near cube) and the bodies
        } else if (t.periodic) { // fp64 monopoles of the coarsest accepted cells + far field -> farc (hot_periodic.cu)
            CUDA_TRY(cudaEventRecord(g.evx[4], st));
            CUDA_TRY(launch_coarse_monopoles(a, t.far, t.farc, g.softening == 1 ? 0.0 : eps * eps, st)); // spline: accepted cells are Newtonian
            a.far = t.farc;
        }
        CUDA_TRY(cudaEventRecord(g.evx[3], st));
        if (!tolmode) {
            CUDA_TRY(launch_forces(a, st));
            if (order > 4) CUDA_TRY(launch_forces_hi(a, order, t.cellHiT, hi_record_floats(t.hi_order), st));
        }
        else { // one launch per order over its part of the cell lists; the first also takes the bodies and the far field
            ForceArgs b = a;
            b.seg = 0; b.order = 0; CUDA_TRY(launch_forces(b, st));
            b.do_pp = 0; b.accumulate = 1; b.far = nullptr;
            for (int sgm = 1; sgm < 3; ++sgm) {
                CUDA_TRY(cudaMemsetAsync(g.d_counter + 1, 0, sizeof(unsigned int), st)); // the work-item scheduler starts over
                b.seg = sgm; b.order = 2 * sgm; CUDA_TRY(launch_forces(b, st));
            }
        }
        CUDA_TRY(cudaEventRecord(g.evx[2], st));
        if (F < ng) { CUDA_TRY(cudaStreamSynchronize(st)); ms_eval += ms_between(g.evx[3], g.evx[2]); if (t.periodic) ms_coarse += ms_between(g.evx[4], g.evx[3]); } // the arena is reused
        if (F < wa.g1) { // the arena was too small: enlarge it if memory allows, else keep going in rounds of what fitted
            const unsigned long long oldpc = cappc, oldpp = cappp;
            cappc *= 2; cappp *= 2;
            rc = clamp_arena(); if (rc) return rc;
            if (cappc < oldpc) cappc = oldpc;
            if (cappp < oldpp) cappp = oldpp;
            if (cappc > oldpc || cappp > oldpp) { rc = alloc_lists(); if (rc) return rc; }
            budget = (F - g0) * (int64_t)((cappc + cappp) / (oldpc + oldpp));
        }
        g.list_g0 = g0; g.list_g1 = F;
        g0 = F;
        ++nrounds;
    }
    CUDA_TRY(launch_group_stats(t.group, t.glpc, t.glpp, t.glvis, tolmode ? t.glpc0 : nullptr, tolmode ? t.glpc2 : nullptr, ng, g.d_stat, st));
    CUDA_TRY(cudaEventRecord(g.ev[7], st));
    unsigned long long stat[6];
    CUDA_TRY(cudaMemcpyAsync(stat, g.d_stat, sizeof(stat), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    ms_eval += ms_between(g.evx[3], g.evx[2]);
    if (t.periodic) ms_coarse += ms_between(g.evx[4], g.evx[3]);
    g.used_pc = usedpc; g.used_pp = usedpp; g.used_groups = ng; // sizes the arena of the next call
    hot_stats_t& s = g.st;
    s.order = order;
    s.cells_visited = stat[0]; s.walk_spills = stat[1]; s.pp_interactions = stat[2]; s.pc_interactions = stat[3];
    s.pc_monopole = s.pc_quadrupole = s.pc_hexadecapole = 0;
    if (tolmode) { s.pc_monopole = stat[4]; s.pc_quadrupole = stat[5]; s.pc_hexadecapole = stat[3] - stat[4] - stat[5]; }
    else (order == 0 ? s.pc_monopole : order == 2 ? s.pc_quadrupole : s.pc_hexadecapole) = stat[3];
    g.last_tolmode = tolmode; g.last_bgmode = bgmode;
    s.ms_moments = ms_between(g.ev[5], g.ev[6]);
    s.ms_walk = ms_walk;
    s.ms_eval = ms_eval;
    s.ms_coarse = ms_coarse;
    s.ms_farfield = ms_between(g.ev[6], g.ev[8]);
    s.ms_forces_total = ms_between(g.ev[5], g.ev[7]);
    s.list_chunks = (int32_t)nrounds; s.list_entries = usedpc + usedpp;
    s.bytes_allocated = g.bytes + (int64_t)g.gstack_bytes;
    s.launches_forces = g_hot_launches;
    g.last_order = order;
    g.lists_valid = true;
    return HOT_OK;
}
} // namespace
extern "C" {
int hot_forces(double theta, double eps, int order, float* acc, float* pot) {
    if (!g.built) return fail(HOT_EORDER, "hot_forces: no successful hot_build");
    if (!acc) return fail(HOT_EINVAL, "hot_forces: NULL acc");
    if (!(theta >= 0.0) || !(theta < 1.0)) return fail(HOT_EINVAL, "hot_forces: theta must be in [0, 1)");
    if (!(eps >= 0.0)) return fail(HOT_EINVAL, "hot_forces: eps must be >= 0");
    if (order != 0 && order != 2 && order != 4 && order != 6 && order != 8) return fail(HOT_EINVAL, "hot_forces: order must be 0, 2, 4, 6 or 8");
    return forces_impl(0, theta, 0.0, eps, order, acc, pot);
}
int hot_forces_tol(double tol, double eps, float* acc, float* pot) {
    if (!g.built) return fail(HOT_EORDER, "hot_forces_tol: no successful hot_build");
    if (!acc) return fail(HOT_EINVAL, "hot_forces_tol: NULL acc");
    if (!(tol >= 0.0) || !(tol < 3.0e38)) return fail(HOT_EINVAL, "hot_forces_tol: tol must be finite and >= 0");
    if (!(eps >= 0.0)) return fail(HOT_EINVAL, "hot_forces_tol: eps must be >= 0");
    return forces_impl(1, 0.0, tol, eps, 4, acc, pot);
}
int hot_export_group_orders(uint64_t* lmono, uint64_t* lquad, uint64_t* lhexa, int64_t cap, int64_t* ngroups) {
    if (!g.built || !g.lists_valid) return fail(HOT_EORDER, "hot_export_group_orders: no hot_forces on this build");
    const Tree& t = g.t;
    if (ngroups) *ngroups = t.ngroups;
    if (cap < t.ngroups) return fail(HOT_EINVAL, "hot_export_group_orders: cap too small");
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    const size_t ng = (size_t)t.ngroups;
    std::vector<uint32_t> tot(ng), a0(ng, 0), a2(ng, 0);
    CUDA_TRY(cudaMemcpy(tot.data(), t.glpc, 4 * ng, cudaMemcpyDeviceToHost));
    if (g.last_tolmode || g.last_bgmode) {
        CUDA_TRY(cudaMemcpy(a0.data(), t.glpc0, 4 * ng, cudaMemcpyDeviceToHost));
        CUDA_TRY(cudaMemcpy(a2.data(), t.glpc2, 4 * ng, cudaMemcpyDeviceToHost));
    }
    if (g.last_bgmode) { // (plain cells, background-subtracted cells, accepted virtual cubes)
        std::vector<uint32_t> pv(ng);
        CUDA_TRY(cudaMemcpy(pv.data(), t.glpv, 4 * ng, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < ng; ++i) {
            if (lmono) lmono[i] = a0[i];
            if (lquad) lquad[i] = a2[i];
            if (lhexa) lhexa[i] = pv[i];
        }
        return HOT_OK;
    } else if (g.last_order == 0) a0 = tot;
    else if (g.last_order == 2) a2 = tot;
    for (size_t i = 0; i < ng; ++i) {
        if (lmono) lmono[i] = a0[i];
        if (lquad) lquad[i] = a2[i];
        if (lhexa) lhexa[i] = (uint64_t)tot[i] - a0[i] - a2[i];
    }
    return HOT_OK;
}

int hot_stats(hot_stats_t* out) {
    if (!out) return fail(HOT_EINVAL, "hot_stats: NULL out");
    *out = g.st;
    return HOT_OK;
}

int hot_step_host(const float* pos, const float* mass, int64_t n, hot_box box, int periodic, double theta, double eps,
                  int order, float* acc, float* pot) {
    if (!pos || !mass || !acc) return fail(HOT_EINVAL, "hot_step_host: NULL argument");
    if (n < 1 || n > ((int64_t)1 << 27)) return fail(HOT_EINVAL, "hot_step_host: n out of range");
    if (g.h_n < n) {
        cudaFree(g.hd_pos); cudaFree(g.hd_mass); cudaFree(g.hd_acc); cudaFree(g.hd_pot);
        g.hd_pos = g.hd_mass = g.hd_acc = g.hd_pot = nullptr; g.h_n = 0;
        CUDA_TRY(cudaMalloc(&g.hd_pos, sizeof(float) * 3 * (size_t)n));
        CUDA_TRY(cudaMalloc(&g.hd_mass, sizeof(float) * (size_t)n));
        CUDA_TRY(cudaMalloc(&g.hd_acc, sizeof(float) * 3 * (size_t)n));
        CUDA_TRY(cudaMalloc(&g.hd_pot, sizeof(float) * (size_t)n));
        g.h_n = n;
    }
    cudaStream_t st = g.stream;
    CUDA_TRY(cudaMemcpyAsync(g.hd_pos, pos, sizeof(float) * 3 * (size_t)n, cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(g.hd_mass, mass, sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, st));
    int rc = hot_build(g.hd_pos, g.hd_mass, n, box, periodic);
    if (rc) return rc;
    // (letting the interaction kernel store into page-locked host arrays directly was measured: 16.7 M scattered 4- and
    // 12-byte writes over PCIe stall it, 144 ms per step against 89 ms with this copy)
    rc = hot_forces(theta, eps, order, g.hd_acc, pot ? g.hd_pot : nullptr);
    if (rc) return rc;
    CUDA_TRY(cudaMemcpyAsync(acc, g.hd_acc, sizeof(float) * 3 * (size_t)n, cudaMemcpyDeviceToHost, st));
    if (pot) CUDA_TRY(cudaMemcpyAsync(pot, g.hd_pot, sizeof(float) * (size_t)n, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return HOT_OK;
}

// ---- introspection -----------------------------------------------------------------------------
int hot_export_keys(uint64_t* key_sorted, uint32_t* perm) {
    if (!g.built) return fail(HOT_EORDER, "hot_export_keys: no build");
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    if (key_sorted) CUDA_TRY(cudaMemcpy(key_sorted, g.t.key[0], sizeof(uint64_t) * (size_t)g.t.n, cudaMemcpyDeviceToHost));
    if (perm) CUDA_TRY(cudaMemcpy(perm, g.t.idx[0], sizeof(uint32_t) * (size_t)g.t.n, cudaMemcpyDeviceToHost));
    return HOT_OK;
}
int hot_export_cells(uint64_t* key, uint32_t* first, uint32_t* count, uint8_t* mask, int32_t* child, int32_t* parent,
                     int64_t cap, int64_t* ncells) {
    if (!g.built) return fail(HOT_EORDER, "hot_export_cells: no build");
    const Tree& t = g.t;
    if (ncells) *ncells = t.ncells;
    if (cap < t.ncells) return fail(HOT_EINVAL, "hot_export_cells: cap %lld < %lld cells", (long long)cap, (long long)t.ncells);
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    size_t nc = (size_t)t.ncells;
    if (key) CUDA_TRY(cudaMemcpy(key, t.ckey, 8 * nc, cudaMemcpyDeviceToHost));
    if (first) CUDA_TRY(cudaMemcpy(first, t.cfirst, 4 * nc, cudaMemcpyDeviceToHost));
    if (count) CUDA_TRY(cudaMemcpy(count, t.ccount, 4 * nc, cudaMemcpyDeviceToHost));
    if (child) CUDA_TRY(cudaMemcpy(child, t.cchild, 4 * nc, cudaMemcpyDeviceToHost));
    if (parent) CUDA_TRY(cudaMemcpy(parent, t.cparent, 4 * nc, cudaMemcpyDeviceToHost));
    if (mask) {
        std::vector<uint32_t> m(nc);
        CUDA_TRY(cudaMemcpy(m.data(), t.cmask, 4 * nc, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nc; ++i) mask[i] = (uint8_t)m[i];
    }
    return HOT_OK;
}
int hot_export_groups(int32_t* cell, uint64_t* key, uint32_t* first, uint32_t* count, uint64_t* lpc, uint64_t* lpp,
                      int64_t cap, int64_t* ngroups) {
    if (!g.built) return fail(HOT_EORDER, "hot_export_groups: no build");
    const Tree& t = g.t;
    if (ngroups) *ngroups = t.ngroups;
    if (cap < t.ngroups) return fail(HOT_EINVAL, "hot_export_groups: cap too small");
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    size_t ng = (size_t)t.ngroups;
    std::vector<GroupRec> r(ng);
    CUDA_TRY(cudaMemcpy(r.data(), t.group, sizeof(GroupRec) * ng, cudaMemcpyDeviceToHost));
    for (size_t i = 0; i < ng; ++i) {
        if (cell) cell[i] = (int32_t)r[i].cell;
        if (first) first[i] = r[i].first;
        if (count) count[i] = r[i].count;
    }
    if (key) {
        std::vector<uint64_t> ck((size_t)t.ncells);
        CUDA_TRY(cudaMemcpy(ck.data(), t.ckey, 8 * (size_t)t.ncells, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < ng; ++i) key[i] = ck[r[i].cell];
    }
    if (lpc || lpp) { // device holds u32 list lengths; L_pp counts the group's own bodies too (they are not in the list)
        std::vector<uint32_t> v(ng);
        if (lpc) {
            CUDA_TRY(cudaMemcpy(v.data(), t.glpc, 4 * ng, cudaMemcpyDeviceToHost));
            for (size_t i = 0; i < ng; ++i) lpc[i] = v[i];
        }
        if (lpp) {
            CUDA_TRY(cudaMemcpy(v.data(), t.glpp, 4 * ng, cudaMemcpyDeviceToHost));
            for (size_t i = 0; i < ng; ++i) lpp[i] = g.lists_valid ? (uint64_t)v[i] + r[i].count : 0;
        }
    }
    return HOT_OK;
}
int hot_export_lists(int64_t group, int32_t* pc_cell, uint8_t* pc_img, int64_t pc_cap, int64_t* npc, uint32_t* pp_body,
                     uint8_t* pp_img, int64_t pp_cap, int64_t* npp) {
    if (!g.built || !g.lists_valid) return fail(HOT_EORDER, "hot_export_lists: no hot_forces on this build");
    const Tree& t = g.t;
    if (!npc || !npp) return fail(HOT_EINVAL, "hot_export_lists: NULL npc / npp");
    if (group < 0 || group >= t.ngroups) return fail(HOT_EINVAL, "hot_export_lists: group %lld outside [0, %lld)", (long long)group, (long long)t.ngroups);
    if (group < g.list_g0 || group >= g.list_g1)
        return fail(HOT_EORDER, "hot_export_lists: the arena holds the lists of groups [%lld, %lld) only", (long long)g.list_g0, (long long)g.list_g1);
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    uint32_t n2[2]; unsigned long long off[2];
    CUDA_TRY(cudaMemcpy(&n2[0], t.glpc + group, 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(&n2[1], t.glpp + group, 4, cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(&off[0], t.pcoff + group, 8, cudaMemcpyDeviceToHost));
    CUDA_TRY(cudaMemcpy(&off[1], t.ppoff + group, 8, cudaMemcpyDeviceToHost));
    *npc = n2[0]; *npp = n2[1];
    if ((pc_cell && pc_cap < (int64_t)n2[0]) || (pc_img && pc_cap < (int64_t)n2[0])) return fail(HOT_EINVAL, "hot_export_lists: pc_cap %lld < %u", (long long)pc_cap, n2[0]);
    if ((pp_body && pp_cap < (int64_t)n2[1]) || (pp_img && pp_cap < (int64_t)n2[1])) return fail(HOT_EINVAL, "hot_export_lists: pp_cap %lld < %u", (long long)pp_cap, n2[1]);
    if (pc_cell && n2[0]) {
        CUDA_TRY(cudaMemcpy(pc_cell, g.d_pclist + off[0], 4 * (size_t)n2[0], cudaMemcpyDeviceToHost));
        for (uint32_t i = 0; i < n2[0]; ++i) pc_cell[i] = (int32_t)((uint32_t)pc_cell[i] & ~HOT_COARSE_FLAG); // the fp64-monopole mark of periodic walks
    }
    if (pp_body && n2[1]) CUDA_TRY(cudaMemcpy(pp_body, g.d_pplist + off[1], 4 * (size_t)n2[1], cudaMemcpyDeviceToHost));
    if (pc_img && n2[0]) { if (t.periodic) CUDA_TRY(cudaMemcpy(pc_img, g.d_pcimg + off[0], n2[0], cudaMemcpyDeviceToHost)); else memset(pc_img, 62, n2[0]); }
    if (pp_img && n2[1]) { if (t.periodic) CUDA_TRY(cudaMemcpy(pp_img, g.d_ppimg + off[1], n2[1], cudaMemcpyDeviceToHost)); else memset(pp_img, 62, n2[1]); }
    return HOT_OK;
}
int hot_export_moments(double* com, float* m0, float* bmax, float* m2, float* m3, float* m4, int64_t cap) {
    if (!g.built || g.t.mom_order < 0) return fail(HOT_EORDER, "hot_export_moments: no hot_forces yet");
    const Tree& t = g.t;
    if (cap < t.ncells) return fail(HOT_EINVAL, "hot_export_moments: cap too small");
    if ((m2 && t.mom_order < 2) || ((m3 || m4) && t.mom_order < 4)) return fail(HOT_EINVAL, "hot_export_moments: order not computed");
    CUDA_TRY(cudaStreamSynchronize(g.stream));
    size_t nc = (size_t)t.ncells;
    if (com || m0 || bmax) {
        std::vector<CellA> a(nc);
        CUDA_TRY(cudaMemcpy(a.data(), t.cellA, sizeof(CellA) * nc, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nc; ++i) {
            if (com) { com[3 * i] = a[i].zx; com[3 * i + 1] = a[i].zy; com[3 * i + 2] = a[i].zz; }
            if (m0) m0[i] = a[i].m0;
            if (bmax) bmax[i] = a[i].bmax;
        }
    }
    if (m2) {
        std::vector<CellM2> a(nc);
        CUDA_TRY(cudaMemcpy(a.data(), t.cellM2, sizeof(CellM2) * nc, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nc; ++i) {
            float* o = m2 + 6 * i;
            o[0] = a[i].xx; o[1] = a[i].xy; o[2] = a[i].xz; o[3] = a[i].yy; o[4] = a[i].yz; o[5] = a[i].zz;
        }
    }
    if (m3 || m4) {
        std::vector<CellM34> a(nc);
        CUDA_TRY(cudaMemcpy(a.data(), t.cellM34, sizeof(CellM34) * nc, cudaMemcpyDeviceToHost));
        for (size_t i = 0; i < nc; ++i) {
            if (m3) memcpy(m3 + 10 * i, a[i].v, 10 * sizeof(float));
            if (m4) memcpy(m4 + 15 * i, a[i].v + 10, 15 * sizeof(float));
        }
    }
    return HOT_OK;
}
int hot_lookup_keys(const uint64_t* keys, int64_t nkeys, int32_t* idx) {
    if (!g.built) return fail(HOT_EORDER, "hot_lookup_keys: no build");
    if (nkeys < 0 || (nkeys > 0 && (!keys || !idx))) return fail(HOT_EINVAL, "hot_lookup_keys: bad arguments");
    if (nkeys == 0) return HOT_OK;
    uint64_t* dk = nullptr; int32_t* di = nullptr;
    CUDA_TRY(cudaMalloc(&dk, 8 * (size_t)nkeys));
    cudaError_t e = cudaMalloc(&di, 4 * (size_t)nkeys);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dk, keys, 8 * (size_t)nkeys, cudaMemcpyHostToDevice, g.stream);
    if (e == cudaSuccess) e = launch_hash_lookup(g.t.ckey, g.t.hval, g.t.hcap - 1, dk, nkeys, di, g.stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(idx, di, 4 * (size_t)nkeys, cudaMemcpyDeviceToHost, g.stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(g.stream);
    cudaFree(dk); cudaFree(di);
    CUDA_TRY(e);
    return HOT_OK;
}

} // extern "C"
