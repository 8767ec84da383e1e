// C ABI of the SABLE B200 library (include/sable.h): context, device upload of the template, launches.
#include "../../include/sable.h"
#include "sable_symbolic.hpp"
#include "sable_kernels2.cuh"

#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace sable;

struct FrontPlan_ { int k = 0, f0 = 0, level = 0; LevelDesc d{}; };
struct sable_ctx {
    Template T;
    sable_options opt{};
    sable_info info{};
    DevTemplate d{};
    std::vector<void*> dev_allocs;
    char* factors = nullptr;  char* work = nullptr;
    int32_t* ints = nullptr;                                 // queue[kMaxChunk] status[mb] it[mb] pivot[mb] active[kMaxActive]
    double* zeros = nullptr;
    const int32_t* fptr = nullptr; const int32_t* fcol = nullptr; const double2* fgb = nullptr;   // full Y_bus, bus order
    const int32_t* ftpos = nullptr; const uint8_t* d_bus_type = nullptr; double* lbuf = nullptr;   // layer backward (lbuf: lazily allocated)
    const int32_t* d_bus_node = nullptr;   // ir_sweeps > 0: node of each bus
    const int32_t* d_long = nullptr; int n_long = 0;   // buses whose Y_bus row has more than 32 entries (warp-served in the bus-order kernels)
    double* irbuf = nullptr;       // ir_sweeps > 0: nine [max_batch][n_bus] arrays (V re/im, |V|, step, residual, correction), allocated at create
    unsigned long long* tim = nullptr;                       // tuning.timing: per-phase cycle counters of CTA 0
    int64_t fac_stride = 0, work_stride = 0;                 // bytes per scenario
    // launch plan of the fused kernel (choose_launch) and of the other kernel families
    int threads = 0, grid = 0, placement = 0, smem = 0, gsh = 0, ctas_per_sm = 1, variant = 0;
    int big_off = 0, slot_off = 0;
    int csz = 1, csz_lin = 1; double* team_red = nullptr;                 // CTAs per team (cluster size) of the fused kernel; per-team norm scratch
    int threads_stage = 0, threads_lin = 0, threads1 = 0;    // staged kernels (group layout), adjoint kernel, one-scenario debug kernels
    int factor_gsh = 0;                                      // group layout of the factors currently in the workspace
    const LevelDesc* level_fused = nullptr; const LevelDesc* level_stage = nullptr;
    const LevelDesc* level_lin = nullptr; const LevelDesc* level_one = nullptr;
    std::vector<LevelDesc> lv_host;                          // blob offsets per level (splits filled per kernel family)
    std::vector<char> blob_host;
    int ring_r = 0, ring_slot = 0, first_staged = 0;
    int front_k = 0, front_f0 = 0, front_level = 0; int64_t front_off = 0; LevelDesc front{};   // dense top front (sable_front.cuh)
    FrontPlan_ lin_front;                                    // the adjoint kernel's own (larger) front
    int last_batch = -1;  bool have_factors = false;
    int64_t launches = 0;
    std::string err;
    // host wrappers: staging buffers (lazily allocated) and the streams / events of the chunk pipeline
    double* hbuf = nullptr; int32_t* hbuf_it = nullptr; uint8_t* hbuf_cv = nullptr;
    cudaStream_t hstream[4] = {nullptr, nullptr, nullptr, nullptr};
};
constexpr int kMaxChunk = 4;      // chunks of the host-buffer pipeline (each with its own queue counter and stream)
constexpr int kMaxActive = 64;    // staged mode: active-scenario counters, one per mismatch pass

static thread_local std::string g_create_err;   // message of the last failed sable_create on this host thread

static sable_status fail(sable_ctx* c, sable_status s, const std::string& m) { if (c) c->err = m; else g_create_err = m; return s; }
#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return fail(ctx, e_ == cudaErrorMemoryAllocation ? SABLE_ERR_ALLOC : SABLE_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); } while (0)

// the library switches to the context's device for the duration of a call and restores the caller's device on return
struct DeviceGuard {
    int prev = -1; cudaError_t err = cudaSuccess;
    explicit DeviceGuard(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev); else if (err == cudaSuccess) prev = -1;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE(ctx) DeviceGuard guard_((ctx)->opt.device); CU(guard_.err)

template <typename V>
static cudaError_t upload(sable_ctx* c, const std::vector<V>& h, const V** out) {
    void* p = nullptr;
    size_t bytes = std::max<size_t>(h.size(), 1) * sizeof(V);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) return e;
    c->dev_allocs.push_back(p);
    if (!h.empty()) e = cudaMemcpy(p, h.data(), h.size() * sizeof(V), cudaMemcpyHostToDevice);
    *out = reinterpret_cast<const V*>(p);
    return e;
}

static void fill_info(sable_ctx* c) {
    const Template& T = c->T;
    sable_info& I = c->info;
    const int64_t w = c->opt.precision == SABLE_MIXED ? 4 : 8;
    I.n_bus = T.n_bus; I.n_pq = T.n_pq; I.n_pv = T.n_pv; I.n = T.n_pv + 2 * T.n_pq;
    I.nnz_y = (int32_t)T.nnz_y; I.nnz_j = (int32_t)T.nnz_j; I.nnz_lu = (int32_t)T.nnz_lu;
    I.n_node = T.n_node; I.n_pair = (int32_t)T.pair_col.size(); I.n_pair_j = (int32_t)T.n_pair_j;
    I.n_level = T.n_level; I.n_term = (int64_t)T.term_a.size(); I.n_term_diag = (int64_t)T.dterm.size();
    I.lu_flops = T.lu_flops;
    I.factor_bytes = (int64_t)(T.n_node + 2 * (int64_t)I.n_pair) * 4 * w;
    // SURVEY.md §8(d) model M0: 8 nnzJ (a2 write) + w nnzJ (a4 read) + 2 w nnzLU (a4 write, a5 read) + 8 (10 nB + 4 n)
    I.bytes_iter_m0 = 8 * T.nnz_j + w * T.nnz_j + 2 * w * T.nnz_lu + 8 * (10 * (int64_t)T.n_bus + 4 * (int64_t)I.n);
    I.bytes_adjoint_m0 = w * T.nnz_lu + 16 * (int64_t)I.n;
    I.smem_bytes = c->smem; I.placement = c->placement; I.threads = c->threads;
    I.ctas_per_sm = c->ctas_per_sm; I.slots_per_cta = 1 << c->gsh; I.cut_level = c->placement == 0 ? 0 : T.n_level;
    I.front_k = c->front_k; I.front_level = c->front_k > 0 ? c->front_level : T.n_level;
    I.threads_lin = c->threads_lin; I.threads_stage = c->threads_stage; I.cluster = c->csz;
}

// kernel variants of the fused kernel: (placement, max threads per CTA, CTAs per SM the registers are budgeted for)
struct Variant { int place, threads, ctas; };
// threads of the CTA that has an SM to itself (register budget 65 536 / kWide, in steps of 8)
#ifndef SABLE_WIDE
#define SABLE_WIDE 768
#endif
constexpr int kWide = SABLE_WIDE;
// CTAs per SM the 128-thread variant is budgeted for: 7 (72 registers) with FP64 factors, kSmallCtasF32 with FP32 factors
template <typename T> struct SmallCtas { static constexpr int v = 7; };
#ifndef SABLE_SMALL_CTAS_F32
#define SABLE_SMALL_CTAS_F32 7
#endif
template <> struct SmallCtas<float> { static constexpr int v = SABLE_SMALL_CTAS_F32; };
static int pick_variant(int place, int th) {
    if (place == 0) return 0;
    return th <= 128 ? 1 : th <= 256 ? 2 : th <= 512 ? 3 : th <= kWide ? 5 : 4;
}
template <typename T> static const void* fused_fn_t(int v) {
    switch (v) {
        case 0: return (const void*)k_nr_fused<T, 0, 512, 1>;
        case 1: return (const void*)k_nr_fused<T, 2, 128, SmallCtas<T>::v>;
        case 2: return (const void*)k_nr_fused<T, 2, 256, 4>;
        case 3: return (const void*)k_nr_fused<T, 2, 512, 2>;
        case 5: return (const void*)k_nr_fused<T, 2, kWide, 1>;
        default: return (const void*)k_nr_fused<T, 2, 1024, 1>;
    }
}
static const void* fused_fn(bool mixed, int v) { return mixed ? fused_fn_t<float>(v) : fused_fn_t<double>(v); }

// threads per CTA of the one-thread-per-bus kernels (recover, layer): whole rounds with no idle tail (300 buses -> 160
// threads x 2 rounds, not 256 x 2 with the second round 85 % idle), 64 for small grids, 512 for large ones
static int bus_threads(int n_bus) {
    if (n_bus <= 256) return 64;
    const int cap = n_bus <= 4096 ? 256 : 512, rounds = (n_bus + cap - 1) / cap;
    return std::min(cap, ((n_bus + rounds - 1) / rounds + 31) / 32 * 32);
}

// A tuning value: the option field if set, else the (debug) environment override, else the default; clamped to [lo, hi].
static int tune(int opt_value, int unset, const char* env, int dflt, int lo, int hi) {
    int v = opt_value != unset ? opt_value : dflt;
    if (opt_value == unset) { const char* e = getenv(env); if (e && *e) v = atoi(e); }
    return std::min(hi, std::max(lo, v));
}
static bool tune_given(int opt_value, int unset, const char* env) { const char* e = getenv(env); return opt_value != unset || (e && *e); }
static int pow2_floor(int x) { int p = 1; while (2 * p <= x) p *= 2; return p; }

// level slices of the index program (layout: LevelDesc in sable_device.cuh).  `d` carries m0, m1, p0, p1; targets are the
// nodes / pairs of that range; only items whose eliminated node k is below k_limit are listed (the front's assembly lists).
struct LevelLists { std::vector<int> dlen, tlen; };   // list lengths in sorted order (for the class cuts)
static LevelLists pack_level(const Template& T, LevelDesc& d, int k_limit, std::vector<char>& blob) {
    auto al = [](size_t x, size_t a) { return (x + a - 1) / a * a; };
    const int nm = d.m1 - d.m0, np = d.p1 - d.p0;
    // item lists per target, filtered
    std::vector<std::vector<int2>> dl(nm);
    std::vector<std::vector<int4>> tl(np);
    for (int i = 0; i < nm; ++i)
        for (int q = T.dterm_ptr[d.m0 + i]; q < T.dterm_ptr[d.m0 + i + 1]; ++q) {
            const int a = T.dterm[q], k = T.pair_row[a];
            if (k < k_limit) dl[i].push_back(make_int2(a, k));
        }
    for (int i = 0; i < np; ++i)
        for (int q = T.term_ptr[d.p0 + i]; q < T.term_ptr[d.p0 + i + 1]; ++q) {
            const int a = T.term_a[q], b = T.term_b[q], k = T.pair_row[a];
            if (k < k_limit) tl[i].push_back(make_int4(a, b, k, 0));
        }
    std::vector<int32_t> dord(nm), tord(np);
    for (int i = 0; i < nm; ++i) dord[i] = i;
    for (int i = 0; i < np; ++i) tord[i] = i;
    std::stable_sort(dord.begin(), dord.end(), [&](int a, int b) { return dl[a].size() > dl[b].size(); });
    std::stable_sort(tord.begin(), tord.end(), [&](int a, int b) { return tl[a].size() > tl[b].size(); });
    size_t nd = 0, nt = 0;
    for (auto& v : dl) nd += v.size();
    for (auto& v : tl) nt += v.size();
    size_t o = 0;
    o += (size_t)(nm + 1) * 4; d.o_dord = (int32_t)o;
    o += (size_t)nm * 4; d.o_tptr = (int32_t)o;
    o += (size_t)(np + 1) * 4; d.o_tord = (int32_t)o;
    o += (size_t)np * 4; d.o_pptr = (int32_t)o;
    o += (size_t)(nm + 1) * 4; o = al(o, 8); d.o_dak = (int32_t)o;
    o += nd * 8; d.o_pmj = (int32_t)o;
    o += (size_t)np * 8; o = al(o, 16); d.o_tab = (int32_t)o;
    o += nt * 16;
    o = al(o, 128);
    d.blob_off = (int32_t)blob.size(); d.blob_bytes = (int32_t)o;
    blob.resize(blob.size() + o, 0);
    char* base = blob.data() + d.blob_off;
    int32_t* dptr = (int32_t*)base; int32_t* dor = (int32_t*)(base + d.o_dord); int32_t* tptr = (int32_t*)(base + d.o_tptr);
    int32_t* tor = (int32_t*)(base + d.o_tord); int32_t* pptr = (int32_t*)(base + d.o_pptr);
    int2* dak = (int2*)(base + d.o_dak); int2* pmj = (int2*)(base + d.o_pmj); int4* tab = (int4*)(base + d.o_tab);
    LevelLists L;
    int32_t q = 0;
    for (int i = 0; i < nm; ++i) {
        dptr[i] = q; dor[i] = dord[i];
        for (const int2& e : dl[dord[i]]) dak[q++] = e;
        L.dlen.push_back((int)dl[dord[i]].size());
    }
    dptr[nm] = q; q = 0;
    for (int i = 0; i < np; ++i) {
        tptr[i] = q; tor[i] = tord[i] | (T.pair_yu[d.p0 + tord[i]] < 0 ? kFromZero : 0);
        for (const int4& e : tl[tord[i]]) tab[q++] = e;
        L.tlen.push_back((int)tl[tord[i]].size());
    }
    tptr[np] = q;
    for (int i = 0; i <= nm; ++i) pptr[i] = T.pair_ptr[d.m0 + i] - d.p0;
    for (int i = 0; i < np; ++i) {
        const int p = d.p0 + i, m = T.pair_row[p], j = T.pair_col[p];
        pmj[i] = make_int2(m | (T.node_pq[m] ? 1 << 30 : 0), j | (T.node_pq[j] ? 1 << 30 : 0));
    }
    return L;
}

// Class cuts of one target kind for a kernel family with `lanes` lanes per slot and at most `wmax` lanes of one warp per
// target: targets are sorted by descending list length `len`; a class is a run of targets that get the same number of
// lanes 2^ssh.  A target asks for enough lanes to leave at most kSerial items per lane; when the level has more lanes than
// its targets ask for, every target gets proportionally more (up to its list length, `boost_max` doublings), so that a narrow
// level spreads over the whole CTA -- in the solve-only sweeps (adjoint kernel); the refactor's levels take no boost (fewer
// lanes per target, shorter shuffle reductions: cfg 5 4.78 -> 4.67 ms, mesh 2.55 -> 2.49, adjoint unchanged).
static int cut_classes(const std::vector<int>& len, int first, int count, int lanes, int wmax, bool diag, int unit, int boost_max, Cls* cls) {
    constexpr int kSerial = 3;      // measured on the B200 (cfg 3 / 4 / 5 / mesh, ms): 1: 2.10 / 3.70 / 5.45 / 2.74; 2: 2.04 / 3.60 / 4.90 / 2.64; 3: 2.02 / 3.63 / 4.74 / 2.55; 4: 2.05 / 3.61 / 4.78 / 2.52
    auto want = [&](int n, int boost) {
        int s = 0;
        while ((1 << s) < wmax && (n + (1 << s) - 1) / (1 << s) > kSerial) ++s;
        while (boost > 0 && (2 << s) <= wmax && (2 << s) <= std::max(1, n)) { ++s; --boost; }
        return s;
    };
    if (count <= 0) return 0;
    int boost = 0;
    for (;; ++boost) {          // largest boost that still fits the CTA in one round
        int64_t need = 0;
        for (int i = first; i < first + count; ++i) need += (int64_t)unit << want(len[i], boost + 1);
        bool grew = false;
        for (int i = first; i < first + count && !grew; ++i) grew = want(len[i], boost + 1) > want(len[i], boost);
        if (need > lanes || !grew || boost >= boost_max) break;
    }
    std::vector<int> ssh(count);
    for (int i = 0; i < count; ++i) ssh[i] = want(len[first + i], boost);
    // at most kMaxCls classes: merge the smallest neighbouring runs upwards (a merged run takes the larger split)
    std::vector<std::pair<int, int>> runs;      // (end index, ssh)
    for (int i = 0; i < count; ++i) {
        if (!runs.empty() && runs.back().second == ssh[i]) runs.back().first = i + 1;
        else runs.push_back({i + 1, ssh[i]});
    }
    while ((int)runs.size() > kMaxCls) {
        int best = 1; int bestlen = 1 << 30;
        for (size_t r = 1; r < runs.size(); ++r) {
            const int l = runs[r].first - runs[r - 1].first;
            if (l < bestlen) { bestlen = l; best = (int)r; }
        }
        runs[best - 1].first = runs[best].first;      // run `best` joins its predecessor (larger or equal split: lists are sorted descending)
        runs.erase(runs.begin() + best);
    }
    int prev = first;
    for (size_t r = 0; r < runs.size(); ++r) {
        cls[r] = Cls{prev * unit, (first + runs[r].first) * unit, (uint8_t)runs[r].second, (uint8_t)(diag ? 1 : 0), 0};
        prev = first + runs[r].first;
    }
    return (int)runs.size();
}

constexpr int kBoostFactor = 0, kBoostSolve = 5;      // lane boost of narrow levels: refactor levels / solve-only sweeps

// lanes per target (log2) for the backward sweep of a level with n targets whose longest list has max_len entries
static uint8_t pick_split(int n, int max_len, int lanes, int wmax) {
    int s = 0;
    while ((2 << s) <= wmax && (int64_t)n * (2 << s) <= lanes && (2 << s) <= std::max(1, max_len)) ++s;
    return (uint8_t)s;
}

// splits / classes of one level descriptor for a kernel family (threads per CTA, slots per CTA)
static void plan_level(const Template& T, LevelDesc& d, const LevelLists& L, int threads, int gsh, bool allow_big, bool staged, int boost_max) {
    const int lanes = std::max(1, threads >> gsh), wmax = std::max(1, 32 >> gsh), nm = d.m1 - d.m0;
    int nbig = 0;
    if (allow_big && lanes >= 2 * wmax) while (nbig < nm && nbig < 4 && L.dlen[nbig] >= 3 * wmax && L.dlen[nbig] >= 64) ++nbig;
    d.n_big = nbig;
    int nc = cut_classes(L.dlen, nbig, nm - nbig, lanes, wmax, true, 1, boost_max, d.cls);
    int with_terms = 0;
    while (with_terms < (int)L.tlen.size() && L.tlen[with_terms] > 0) ++with_terms;
    nc += cut_classes(L.tlen, 0, with_terms, lanes, wmax, false, kTargetUnit, boost_max, d.cls + nc);
    d.n_cls = (uint8_t)nc;
    int maxb = 0;
    for (int m = d.m0; m < d.m1; ++m) maxb = std::max(maxb, T.pair_ptr[m + 1] - T.pair_ptr[m]);
    d.sb = pick_split(nm, maxb, lanes, wmax);
    d.staged = staged;
}

struct LevelPack { std::vector<LevelDesc> lv; std::vector<LevelLists> lists; };

static std::vector<LevelDesc> build_levels(const Template& T, const LevelPack& P, int threads, int gsh, bool allow_big, int first_staged, int boost_max) {
    std::vector<LevelDesc> lv(P.lv);
    for (int l = 0; l < T.n_level; ++l) plan_level(T, lv[l], P.lists[l], threads, gsh, allow_big, l >= first_staged, boost_max);
    return lv;
}

// Dense top front (sable_front.cuh): the nodes of the last elimination levels, as many levels as keep the K x K block
// matrix within `budget` bytes of shared memory per CTA (K <= kcap).  Appends the assembly lists (the front targets'
// items whose eliminated node k lies below the front) to the blob and fills ctx->front*.
struct FrontPlan { int k = 0, f0 = 0, level = 0; LevelDesc d{}; };
static FrontPlan build_front(sable_ctx* c, int threads, int gsh, int64_t budget, int kcap, bool allow_big, int boost_max) {
    const Template& T = c->T;
    const int nn = T.n_node, np = (int)T.pair_col.size(), nl = T.n_level;
    const bool mixed = c->opt.precision == SABLE_MIXED;
    FrontPlan fp; fp.k = 0; fp.f0 = nn; fp.level = nl;
    auto bytes = [&](int K) { return mixed ? front_bytes<float>(K, gsh) : front_bytes<double>(K, gsh); };
    int lc = nl;
    while (lc > 1 && nn - T.level_ptr[lc - 1] <= kcap && bytes(nn - T.level_ptr[lc - 1]) <= budget) --lc;
    if (nl - lc < 2) return fp;                              // merging fewer than two levels saves nothing
    const int f0 = T.level_ptr[lc];
    LevelDesc d{};
    d.m0 = f0; d.m1 = nn; d.p0 = T.pair_ptr[f0]; d.p1 = np;
    const LevelLists L = pack_level(T, d, f0, c->blob_host);
    plan_level(T, d, L, threads, gsh, allow_big, false, boost_max);
    fp.d = d; fp.k = nn - f0; fp.f0 = f0; fp.level = lc;
    return fp;
}

// Launch plan of the fused kernel (DESIGN.md "Placement" and "Launch policy").
static sable_status choose_launch(sable_ctx* ctx, const LevelPack& P) {
    const Template& T = ctx->T;
    const sable_tuning& tu = ctx->opt.tune;
    const int nn = T.n_node, np = (int)T.pair_col.size(), nl = T.n_level;
    const bool mixed = ctx->opt.precision == SABLE_MIXED;
    int dev = 0; CU(cudaGetDevice(&dev));
    int max_optin = 0, n_sm = 0, smem_sm = 0;
    CU(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    CU(cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    const int mb = ctx->opt.max_batch;
    int ring_bytes = 0;
    auto need = [&](int th, int gsh, bool on_chip) {
        const int big = (int)big_bytes(th, gsh);
        return mixed ? smem_need<float>(nn, np, nl, ring_bytes, big, gsh, on_chip) : smem_need<double>(nn, np, nl, ring_bytes, big, gsh, on_chip);
    };
    // ring candidates (slots, slot capacity): the streamed levels are the trailing run of levels whose blobs fit a slot
    struct RingOpt { int r, cap; };
    const bool ring_given = tune_given(tu.ring_slots, -1, "SABLE_RING_R") || tune_given(tu.ring_slot_bytes, -1, "SABLE_RING_SLOT");
    std::vector<RingOpt> ropts = {{3, 8192}, {2, 8192}, {3, 4096}, {2, 4096}, {2, 2048}, {0, 0}};
    if (ring_given) ropts = {{tune(tu.ring_slots, -1, "SABLE_RING_R", 3, 0, kMaxRing), tune(tu.ring_slot_bytes, -1, "SABLE_RING_SLOT", 8192, 256, 65536) / 16 * 16}, {0, 0}};
    auto set_ring = [&](const RingOpt& o) {
        int first = nl, slot = 0;
        if (o.r > 0) while (first > 0 && P.lv[first - 1].blob_bytes <= o.cap) { --first; slot = std::max(slot, P.lv[first].blob_bytes); }
        if (first == nl) { ctx->ring_r = 0; ctx->ring_slot = 0; ctx->first_staged = nl; ring_bytes = 0; return; }
        ctx->ring_r = o.r; ctx->ring_slot = slot; ctx->first_staged = first; ring_bytes = o.r * slot;
    };
    const bool th_given = ctx->opt.threads > 0 || tune_given(0, 0, "SABLE_THREADS");
    const bool g_given = tune_given(tu.group, 0, "SABLE_G");
    const int g_want = pow2_floor(tune(tu.group, 0, "SABLE_G", 1, 1, 32));
    const int want_chip = tune(tu.on_chip, -1, "SABLE_ONCHIP", -1, -1, 1);
    // ---- on-chip candidate: as many scenario slots per CTA as fit entirely in shared memory (G = 8, 4, 2, 1) ----------
    int th0 = ctx->opt.threads > 0 ? ctx->opt.threads : nn <= 64 ? 64 : nn <= 200 ? 256 : 512;
    th0 = std::min(512, std::max(32, (tune(0, 0, "SABLE_THREADS", th0, 32, 512) + 31) / 32 * 32));
    int gsh0 = -1;
    for (int cand = 3; cand >= 0 && gsh0 < 0 && want_chip != 0; --cand) {
        if (g_given && (1 << cand) != g_want) continue;
        // do not group more scenarios per CTA than leaves every SM a CTA (small batches stay spread out)
        if (!g_given && cand > 0 && (int64_t)n_sm * (1 << cand) > (int64_t)mb) continue;
        if ((th0 >> cand) < 8) continue;
        // the blob ring pays only where the slots leave no L1 for the index program (measured in round 1: cfg 2 with
        // 57 KB of L1 left runs 0.133 ms without the ring, 0.147 ms with it; cfg 3 on chip with 21 KB left 4.9 vs 4.4 ms)
        if (!ring_given) {
            set_ring(RingOpt{0, 0});
            const int64_t n0 = need(th0, cand, true) + 1024;
            if (n0 <= max_optin && smem_sm - (smem_sm / n0) * n0 >= 32 * 1024) { gsh0 = cand; break; }
        }
        for (const RingOpt& o : ropts) {
            set_ring(o);
            if (need(th0, cand, true) <= max_optin) { gsh0 = cand; break; }
        }
    }
    // all on chip only while the SMs can hold a good part of the batch at once; a batch of many waves runs faster from
    // the group-interleaved HBM workspace with many small CTAs (round 1: cfg 3 3.5 ms vs 4.4 ms)
    bool on_chip = gsh0 >= 0;
    if (on_chip && want_chip < 0) {
        const int64_t slots_sm = (int64_t)std::max<int64_t>(1, smem_sm / (need(th0, gsh0, true) + 1024)) << gsh0;
        if (slots_sm * n_sm * 2 < (int64_t)mb) on_chip = false;
    }
    int th, gsh;
    if (on_chip) {
        ctx->placement = 0; th = th0; gsh = gsh0; ctx->csz = 1;
    } else {
        // ---- HBM placement (everything in the group-interleaved workspace, blobs read in place, no ring) --------------
        // Occupancy model.  The path is bound by memory latency: the SM should hold as many
        // independent elimination chains (scenarios) as its registers allow, each with enough lanes for its levels.
        //  * lanes per scenario L: 0.75 x the mean number of multiply-subtract items of an elimination level, as a power of
        //    two in [16, 512] -- a tree-like 300-bus grid gets 16 (2.05 ms against 2.15 at 32), a 2 000-bus grid 128, a 900-bus mesh with 3x fill 256, the
        //    9 241-bus grid 512 (each measured best: 3.83 vs 4.03 ms at 256 on the 2 000-bus grid, 4.1 vs 5.2 ms at 128 on the mesh);
        //  * slots per CTA G such that a CTA has about 128 threads (small CTAs pack the register file best: 7 x 128 at 72
        //    registers), never so many that the batch leaves SMs without a CTA;
        //  * single-wave batches (2 / 4 / 8 / 16 scenarios per SM fill the SMs in one wave: 256 scenarios of 9 241 buses, 512 of
        //    the 900-bus mesh, 2 048 of 2 000 buses): the CTAs that would share an SM anyway are merged into ONE CTA of 768
        //    (1 024) threads whose scenarios interleave their slices -- neighbouring lanes then read neighbouring words (a
        //    fraction of the L1 wavefronts: 6.2 vs 6.6 ms on the 9 241-bus grid, 2.63 vs 3.56 on the mesh, 3.63 vs 3.93 on
        //    the 2 000-bus grid with FP32 factors);
        //  * teams (a cluster of CTAs per group): for tiny batches of large grids (below), or on request (tune.cluster).
        const double items = (double)T.term_a.size() + (double)T.dterm.size();
        const int L = std::min(512, std::max(16, pow2_floor(std::max(1, (int)(0.75 * items / std::max(1, nl))))));
        const int c_given = tune_given(tu.cluster, 0, "SABLE_CLUSTER");
        int csz = c_given ? pow2_floor(tune(tu.cluster, 0, "SABLE_CLUSTER", 1, 1, 8)) : 1;
        int G = std::max(1, 128 / L);
        bool merged = false;
        if (g_given) G = g_want;
        else {
            while (G > 1 && (int64_t)n_sm * G > (int64_t)std::max(mb, 1)) G /= 2;
            // merged single-wave layout: when g = 2 / 4 / 8 / 16 scenarios per SM make one wave that still fills the SMs (at
            // least 85 % of them get a group), the g CTAs that would share an SM become ONE CTA whose g scenarios interleave
            for (int g = 2 * G; g <= 16 && !merged; g *= 2) {
                const int64_t groups = ((int64_t)mb + g - 1) / g;
                if (groups <= n_sm && 20 * groups >= 17 * (int64_t)n_sm) { G = g; merged = true; }
            }
        }
        // tiny batches of large grids (the paper's own shapes: 4 ... 32 scenarios of 9 241 buses): the scenarios cannot fill
        // the SMs, and one scenario's wide levels want more lanes than a CTA has -- a team of 2 / 4 / 8 CTAs (one cluster) per
        // scenario, as large as keeps all teams within half of the SMs (clusters are placed GPC by GPC).  Measured on the
        // only the very large grids gain: see below.
        if (!c_given && !g_given && !th_given && ctx->opt.threads <= 0 && G == 1 && L >= 512 && nn >= 16384)
            while (csz < 8 && (int64_t)mb * csz * 2 * 2 <= n_sm) csz *= 2;
        // batches that leave every CTA an SM of its own: the CTA takes 768 threads (and the large front budget below) whatever
        // the grid -- 9 241-bus stand-in, 64 scenarios: 4.14 ms at 256 threads, 2.46 at 768; 3 120 buses x 8: 2.05 -> 1.29;
        // 1 354 buses x 8: 0.79 -> 0.60 (a team of CTAs per scenario is slower there: 2.40 ms for 4 scenarios of 9 241 buses
        // against 2.28; it wins on the 25 000-bus stand-in, 27 vs 33 ms for 8 scenarios x 30 iterations)
        const bool alone = (int64_t)(mb + G - 1) / G <= n_sm && G == 1;
        gsh = 0; while ((2 << gsh) <= G) ++gsh;
        // (the merged layout runs 768 threads, 80 registers each: 5.35 ms against 5.63 at 1 024 threads / 64 registers)
        // (a merged CTA wants at least 64 lanes per scenario: 1 024 threads for 16 scenarios, 768 otherwise)
        th = ctx->opt.threads > 0 ? ctx->opt.threads : csz > 1 ? 1024 : merged ? (kWide >> gsh >= 64 ? kWide : 1024)
                                                                              : (alone || (L << gsh) >= 1024) ? kWide : (L << gsh);
        th = std::min(1024, std::max(32, (tune(0, 0, "SABLE_THREADS", th, 32, 1024) + 31) / 32 * 32));
        if ((th >> gsh) < 1) gsh = 0;
        ctx->placement = 2; ctx->csz = csz;
        set_ring(RingOpt{0, 0});
        if (need(th, gsh, false) > max_optin) return fail(ctx, SABLE_ERR_INVALID_ARG, "placement does not fit shared memory");
    }
    ctx->threads = th; ctx->gsh = gsh;
    ctx->variant = pick_variant(ctx->placement, th);
    const int big = (int)big_bytes(th, gsh);
    ctx->big_off = (int)(smem_fixed(nl, ring_bytes, 0));
    ctx->slot_off = (int)smem_fixed(nl, ring_bytes, big);
    ctx->smem = (int)need(th, gsh, on_chip);
    ctx->front_k = 0; ctx->front_level = nl; ctx->front_f0 = nn;
    if (ctx->placement == 2) {
        // dense top front: shared memory that still leaves most of the L1 to the resident CTAs
        const int kcap = tune(tu.front_nodes, -1, "SABLE_FRONT", 64, 0, 96);
        // (a CTA that has the SM to itself -- the merged single-wave layout -- can afford a large front: 5.69 ms with 32 nodes
        // against 5.98 with 15 and 6.17 without on the 9 241-bus grid; small CTAs that share the SM keep the L1)
        const int64_t budget = tune(tu.front_kb, -1, "SABLE_FRONT_KB", th <= 128 ? 8 : th <= 256 ? 6 : th <= 512 ? 16 : 96, 0, 220) * 1024LL;
        if (kcap >= 2 && ctx->csz == 1) {
            const FrontPlan fp = build_front(ctx, th, gsh, budget, kcap, true, kBoostFactor);
            ctx->front = fp.d; ctx->front_k = fp.k; ctx->front_f0 = fp.f0; ctx->front_level = fp.level;
        }
        if (ctx->front_k > 0) {
            ctx->front_off = align16(ctx->smem);
            ctx->smem = (int)(ctx->front_off + (mixed ? front_bytes<float>(ctx->front_k, gsh) : front_bytes<double>(ctx->front_k, gsh)));
        }
    }
    if (ctx->smem > max_optin) return fail(ctx, SABLE_ERR_INVALID_ARG, "launch plan does not fit shared memory");
    const void* fn = fused_fn(mixed, ctx->variant);
    CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, th, (size_t)ctx->smem));
    if (occ < 1) return fail(ctx, SABLE_ERR_CUDA, "NR kernel does not fit on an SM");
    occ = std::min(occ, tune(tu.ctas_per_sm, 0, "SABLE_CTAS", occ, 1, 32));
    ctx->ctas_per_sm = occ; ctx->grid = occ * n_sm / ctx->csz * ctx->csz;
    // the other kernel families: staged kernels (same group layout; the fused kernel's own shape when it is an HBM kernel),
    // the adjoint kernel (32 targets in flight per slot measured best in round 1), one-scenario debug kernels
    const int Ls = std::min(512, std::max(32, pow2_floor(std::max(1, nn / 8))));
    ctx->threads_stage = (tune(tu.threads_stage, 0, "SABLE_THREADS1", ctx->placement == 2 ? th : std::min(512, Ls << gsh), 32, 1024) + 31) / 32 * 32;
    ctx->csz_lin = ctx->csz;
    // adjoint kernel: 32 lanes per slot (measured best in round 1: a pure latency chain wants many small CTAs); the merged
    // single-wave layout (two slots of a large grid per CTA) wants the whole SM
    ctx->threads_lin = (tune(tu.threads_lin, 0, "SABLE_THREADS_LIN", ctx->csz > 1 ? 512 : (gsh >= 1 && th >= kWide) ? 1024 : std::min(512, std::max(32 << gsh, 64)), 32, 1024) + 31) / 32 * 32;
    ctx->threads1 = nn <= 64 ? 32 : nn <= 1200 ? 64 : nn <= 4000 ? 256 : 512;
    // the adjoint kernel's dense front: its shared memory holds nothing else of size, so when every CTA has an SM of its own
    // the front takes up to 180 KB (9 241-bus grid: 54 nodes instead of the NR kernel's 38); otherwise the NR kernel's front
    ctx->lin_front = FrontPlan_{ctx->front_k, ctx->front_f0, ctx->front_level, ctx->front};
    if (ctx->placement == 2 && ctx->csz == 1 && ctx->front_k > 0 && (int64_t)((mb + (1 << gsh) - 1) >> gsh) <= n_sm &&
        !tune_given(tu.front_kb, -1, "SABLE_FRONT_KB") && !tune_given(tu.front_nodes, -1, "SABLE_FRONT")) {
        const FrontPlan fp = build_front(ctx, ctx->threads_lin, gsh, 180 * 1024LL, 96, true, kBoostSolve);
        if (fp.k > ctx->front_k) ctx->lin_front = FrontPlan_{fp.k, fp.f0, fp.level, fp.d};
    }
    return SABLE_OK;
}

extern "C" sable_status sable_create(int32_t n_bus, const int32_t* row_ptr, const int32_t* col_idx, const double* y_re,
                                     const double* y_im, const uint8_t* bus_type, int32_t slack,
                                     const sable_options* opt, sable_ctx** out) {
    sable_ctx* ctx = nullptr;      // CU() reports into g_create_err while ctx is null
    if (!out) return fail(nullptr, SABLE_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    sable_options o = sable_default_options();
    if (opt) o = *opt;
    if (o.max_batch < 1 || (o.precision != SABLE_FP64 && o.precision != SABLE_MIXED) ||
        (o.mode != SABLE_MODE_FUSED && o.mode != SABLE_MODE_STAGED) || o.device < -1 || o.threads < 0 || o.ir_sweeps < 0 || o.ir_sweeps > 8)
        return fail(nullptr, SABLE_ERR_INVALID_ARG, "bad option value");
    if (o.ir_sweeps > 0 && (o.precision != SABLE_MIXED || o.mode != SABLE_MODE_STAGED))
        return fail(nullptr, SABLE_ERR_INVALID_ARG, "ir_sweeps > 0 needs precision = SABLE_MIXED (FP32 factors to refine) and mode = SABLE_MODE_STAGED "
                    "(the sweeps run as kernels of their own between the solve stage and the update)");
    sable_ctx* c = new (std::nothrow) sable_ctx;
    if (!c) return fail(nullptr, SABLE_ERR_ALLOC, "host allocation failed");
    c->opt = o;
    std::string err;
    int rc = build_template(n_bus, row_ptr, col_idx, y_re, y_im, bus_type, slack, c->T, err);
    if (rc) { delete c; return fail(nullptr, (sable_status)rc, err); }
    if (o.device < 0) { fill_info(c); *out = c; return SABLE_OK; }

    const Template& T = c->T;
    const int nn = T.n_node, np = (int)T.pair_col.size();
    auto bail = [&](sable_status s) { std::string m = c->err; sable_destroy(c); g_create_err = m; return s; };
    DeviceGuard guard(o.device);
    if (guard.err != cudaSuccess) { c->err = std::string("cudaSetDevice: ") + cudaGetErrorString(guard.err); return bail(SABLE_ERR_CUDA); }
    // packed device arrays
    std::vector<int32_t> node_bus(T.node_bus); node_bus.push_back(T.slack);
    std::vector<double2> ygb(T.ycol.size()), ydg(nn);
    for (size_t k = 0; k < T.ycol.size(); ++k) ygb[k] = make_double2(T.yg[k], T.yb[k]);
    for (int m = 0; m < nn; ++m) ydg[m] = make_double2(T.yg[T.ydiag[m]], T.yb[T.ydiag[m]]);
    // Jacobian destinations of the Y entries (stage_mismatch): entry (m,j) of row m feeds the U half of pair (m,j) when j is
    // eliminated later, the L' half of pair (j,m) otherwise; diagonal entries and the slack column feed nothing
    std::vector<int2> ycd(T.ycol.size());
    std::vector<int4> jmj;
    std::vector<double4> jy;
    for (size_t k = 0; k < T.ycol.size(); ++k) ycd[k] = make_int2(T.ycol[k], -1);
    for (int p = 0; p < np; ++p) {
        const int su = T.pair_yu[p], sl = T.pair_yl[p];
        if ((su >= 0) != (sl >= 0)) { c->err = "internal: Y pattern not symmetric"; return bail(SABLE_ERR_STRUCTURE); }
        if (su < 0) continue;
        ycd[su].y = p | (T.node_pq[T.pair_col[p]] ? 1 << 30 : 0);
        const int m = T.pair_row[p], j = T.pair_col[p];
        jmj.push_back(make_int4(m | (T.node_pq[m] ? 1 << 30 : 0), j | (T.node_pq[j] ? 1 << 30 : 0), p, 0));
        jy.push_back(make_double4(T.yg[su], T.yb[su], T.yg[sl], T.yb[sl]));
        ycd[sl].y = p | 1 << 29 | (T.node_pq[T.pair_row[p]] ? 1 << 30 : 0);
    }
    DevTemplate& d = c->d;
    d.n_bus = T.n_bus; d.n_node = nn; d.n_pair = np; d.n_level = T.n_level; d.slack = T.slack;
    // mismatch pass: nodes by descending Y-row length; a row of up to 12 << s entries is served by 1 << s lanes
    std::vector<int32_t> mm_order(nn);
    std::vector<int4> mm_row(nn);
    {
        for (int m = 0; m < nn; ++m) mm_order[m] = m;
        auto deg = [&](int m) { return T.yptr[m + 1] - T.yptr[m]; };
        std::stable_sort(mm_order.begin(), mm_order.end(), [&](int a, int b) { return deg(a) > deg(b); });
        auto cls = [&](int m) { int sft = 0; while (sft < 5 && deg(m) > (12 << sft)) ++sft; return sft; };
        d.n_class = 0;
        for (int i = 0; i < nn;) {
            int j = i; const int sft = cls(mm_order[i]);
            while (j < nn && cls(mm_order[j]) == sft) ++j;
            d.mm_class[d.n_class++] = RowClass{i, j, sft};
            i = j;
        }
        for (int i = 0; i < nn; ++i) {
            const int m = mm_order[i];
            mm_row[i] = make_int4(m, T.yptr[m], T.yptr[m + 1], T.node_bus[m] | (T.node_pq[m] ? 1 << 30 : 0));
        }
    }
    bool ok = true;
    auto up = [&](auto& vec, auto** dst) { if (ok && upload(c, vec, dst) != cudaSuccess) { ok = false; c->err = "template upload failed"; } };
    {
        std::vector<double2> fgb(T.fcol.size());
        for (size_t k = 0; k < fgb.size(); ++k) fgb[k] = make_double2(T.fg[k], T.fb[k]);
        up(T.fptr, &c->fptr); up(T.fcol, &c->fcol); up(fgb, &c->fgb);
        std::vector<int32_t> tpos(T.fcol.size());
        for (int i = 0; i < T.n_bus; ++i)
            for (int k = T.fptr[i]; k < T.fptr[i + 1]; ++k) {
                const int j = T.fcol[k];
                auto bj = T.fcol.begin() + T.fptr[j], ej = T.fcol.begin() + T.fptr[j + 1];
                tpos[k] = (int32_t)(std::lower_bound(bj, ej, i) - T.fcol.begin());   // the pattern is symmetric (canonicalised)
            }
        std::vector<uint8_t> bt(bus_type, bus_type + n_bus);
        up(tpos, &c->ftpos); up(bt, &c->d_bus_type);
        if (o.ir_sweeps > 0) up(T.bus_node, &c->d_bus_node);
        std::vector<int32_t> longr;
        for (int i = 0; i < T.n_bus; ++i) if (T.fptr[i + 1] - T.fptr[i] > 32) longr.push_back(i);
        c->n_long = (int)longr.size();
        if (c->n_long) up(longr, &c->d_long);
    }
    up(mm_row, &d.mm_row); up(node_bus, &d.node_bus); up(T.node_pq, &d.node_pq); up(T.yptr, &d.yptr);
    up(T.ycol, &d.ycol); up(ycd, &d.ycd); up(ygb, &d.ygb); up(jmj, &d.jp_mj); up(jy, &d.jp_y);
    d.n_jpair = (int)jmj.size(); up(ydg, &d.ydiag_gb);
    if (!ok) return bail(SABLE_ERR_ALLOC);
    ctx = c;
    LevelPack P;
    P.lv.assign(T.n_level, LevelDesc{});
    for (int l = 0; l < T.n_level; ++l) {
        LevelDesc& ld = P.lv[l];
        ld.m0 = T.level_ptr[l]; ld.m1 = T.level_ptr[l + 1]; ld.p0 = T.pair_ptr[ld.m0]; ld.p1 = T.pair_ptr[ld.m1];
        P.lists.push_back(pack_level(T, ld, nn, c->blob_host));
    }
    c->lv_host = P.lv;
    sable_status st = choose_launch(c, P);
    if (st != SABLE_OK) return bail(st);
    {
        std::vector<LevelDesc> lf = build_levels(T, P, c->threads * c->csz, c->gsh, c->csz == 1, c->first_staged, c->placement == 2 ? kBoostFactor : kBoostSolve);
        std::vector<LevelDesc> ls = build_levels(T, P, c->threads_stage, c->gsh, ((c->threads_stage >> 5) << c->gsh) <= 256, T.n_level, kBoostFactor);
        std::vector<LevelDesc> ll = build_levels(T, P, c->threads_lin * c->csz_lin, c->gsh, c->csz_lin == 1, T.n_level, kBoostSolve);
        std::vector<LevelDesc> l1 = build_levels(T, P, c->threads1, 0, true, T.n_level, kBoostSolve);
        up(lf, &c->level_fused); up(ls, &c->level_stage); up(ll, &c->level_lin); up(l1, &c->level_one); up(c->blob_host, &d.blob);
        if (!ok) return bail(SABLE_ERR_ALLOC);
    }
    const bool mixed = o.precision == SABLE_MIXED;
    c->fac_stride = ((mixed ? fac_bytes<float>(nn, np) + 16 : fac_bytes<double>(nn, np)) + 31) & ~int64_t(31);   // whole 32-byte units (FP32: room for the alignment of the pair records)
    c->work_stride = work_bytes(nn);
    auto dmalloc = [&](void** p, size_t bytes) {
        if (cudaMalloc(p, bytes) != cudaSuccess) { c->err = "device allocation failed (" + std::to_string(bytes) + " bytes)"; return false; }
        c->dev_allocs.push_back(*p); return true;
    };
    const size_t mb = (size_t)o.max_batch, nb = (size_t)T.n_bus;
    // workspace for whole groups of 1 << gsh scenarios + one spare group that absorbs the stores of finished slots
    const size_t G = (size_t)1 << c->gsh, mb_alloc = (mb + G - 1) / G * G + G;
    const size_t n_ints = kMaxChunk + 3 * mb + kMaxActive;
    if (!dmalloc((void**)&c->factors, mb_alloc * c->fac_stride) || !dmalloc((void**)&c->work, mb_alloc * c->work_stride) ||
        !dmalloc((void**)&c->ints, n_ints * 4) || !dmalloc((void**)&c->zeros, nb * 8) ||
        !dmalloc((void**)&c->team_red, (size_t)kMaxChunk * std::max(1, c->grid) * G * 8))
        return bail(SABLE_ERR_ALLOC);
    if (cudaMemset(c->zeros, 0, nb * 8) != cudaSuccess || cudaMemset(c->work, 0, mb_alloc * c->work_stride) != cudaSuccess ||
        cudaMemset(c->factors, 0, mb_alloc * c->fac_stride) != cudaSuccess || cudaMemset(c->ints, 0, n_ints * 4) != cudaSuccess) {
        c->err = "cudaMemset failed"; return bail(SABLE_ERR_CUDA);
    }
    if (tune(o.tune.timing, 0, "SABLE_TIMING", 0, 0, 1)) {
        const size_t tb = (4 * (size_t)T.n_level + 4) * 8;
        if (!dmalloc((void**)&c->tim, tb)) return bail(SABLE_ERR_ALLOC);
        cudaMemset(c->tim, 0, tb);
    }
    if (o.ir_sweeps > 0) {                                   // sable_solve itself allocates nothing
        const size_t ib = 9 * (size_t)o.max_batch * nb * 8;
        if (!dmalloc((void**)&c->irbuf, ib)) return bail(SABLE_ERR_ALLOC);
        if (cudaMemset(c->irbuf, 0, ib) != cudaSuccess) { c->err = "cudaMemset failed"; return bail(SABLE_ERR_CUDA); }
    }
    fill_info(c);
    *out = c;
    return SABLE_OK;
}

extern "C" sable_options sable_default_options(void) {
    sable_options o{};
    o.max_batch = 1; o.precision = SABLE_FP64; o.keep_factors = 1; o.mode = SABLE_MODE_FUSED; o.device = 0; o.threads = 0; o.ir_sweeps = 0;
    o.tune.group = 0; o.tune.ctas_per_sm = 0; o.tune.on_chip = -1; o.tune.ring_slots = -1; o.tune.ring_slot_bytes = -1;
    o.tune.front_nodes = -1; o.tune.front_kb = -1; o.tune.threads_stage = 0; o.tune.threads_lin = 0; o.tune.timing = 0; o.tune.cluster = 0;
    return o;
}

extern "C" void sable_destroy(sable_ctx* c) {
    if (!c) return;
    if (c->opt.device >= 0) {
        DeviceGuard guard(c->opt.device);
        for (cudaStream_t s : c->hstream) if (s) cudaStreamDestroy(s);
        for (void* p : c->dev_allocs) cudaFree(p);
    }
    delete c;
}
extern "C" const char* sable_last_error(const sable_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }
extern "C" int64_t sable_launch_count(const sable_ctx* c) { return c ? c->launches : 0; }
extern "C" sable_status sable_get_info(const sable_ctx* c, sable_info* info) {
    if (!c || !info) return SABLE_ERR_INVALID_ARG;
    *info = c->info; return SABLE_OK;
}

// ---- solve -------------------------------------------------------------------------------------------------------
static int32_t* ctx_status(sable_ctx* c) { return c->ints + kMaxChunk; }
static int32_t* ctx_it(sable_ctx* c) { return c->ints + kMaxChunk + c->opt.max_batch; }
static int32_t* ctx_pivot(sable_ctx* c) { return c->ints + kMaxChunk + 2 * (size_t)c->opt.max_batch; }
static int32_t* ctx_active(sable_ctx* c) { return c->ints + kMaxChunk + 3 * (size_t)c->opt.max_batch; }

template <typename T>
static cudaError_t launch_fused(sable_ctx* c, const SolveArgs& A, cudaStream_t s) {
    const int G = 1 << c->gsh, groups = (A.batch + G - 1) / G;
    const int grid = std::min(groups, std::max(1, c->grid / c->csz)) * c->csz;     // whole teams
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(c->threads); cfg.dynamicSmemBytes = (size_t)c->smem; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = c->csz; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = c->csz > 1 ? 1 : 0;
    switch (c->variant) {
        case 0: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 0, 512, 1>, A);
        case 1: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 2, 128, SmallCtas<T>::v>, A);
        case 2: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 2, 256, 4>, A);
        case 3: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 2, 512, 2>, A);
        case 5: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 2, kWide, 1>, A);
        default: return cudaLaunchKernelEx(&cfg, k_nr_fused<T, 2, 1024, 1>, A);
    }
}

// staged kernels: the instantiation whose register budget fits the thread count
template <typename T> static void launch_st_mismatch_fill(const SolveArgs& A, int grid, int th, cudaStream_t s) {
    if (th <= 128) k_st_mismatch_fill<T, 128, 7><<<grid, th, 0, s>>>(A);
    else if (th <= 512) k_st_mismatch_fill<T, 512, 2><<<grid, th, 0, s>>>(A);
    else if (th <= kWide) k_st_mismatch_fill<T, kWide, 1><<<grid, th, 0, s>>>(A);
    else k_st_mismatch_fill<T, 1024, 1><<<grid, th, 0, s>>>(A);
}
template <typename T> static void launch_st_factor_solve(const SolveArgs& A, int grid, int th, cudaStream_t s) {
    if (th <= 128) k_st_factor_solve<T, 128, 7><<<grid, th, 0, s>>>(A);
    else if (th <= 512) k_st_factor_solve<T, 512, 2><<<grid, th, 0, s>>>(A);
    else if (th <= kWide) k_st_factor_solve<T, kWide, 1><<<grid, th, 0, s>>>(A);
    else k_st_factor_solve<T, 1024, 1><<<grid, th, 0, s>>>(A);
}

static sable_status launch_lin(sable_ctx* ctx, int b0, int batch, const double* rp, const double* rq, int transposed, double* xp,
                               double* xq, bool use_flags, cudaStream_t s);

// Scenarios [b0, b0 + nb) of the caller's arrays (b0 a multiple of the group size) on stream s, with queue counter `chunk`.
template <typename T>
static cudaError_t launch_solve(sable_ctx* c, SolveArgs A, int b0, int nb, int chunk, cudaStream_t s) {
    const size_t o = (size_t)b0 * c->T.n_bus;
    const int G = 1 << c->gsh, g0 = b0 >> c->gsh;
    A.batch = nb;
    A.p_spec += o; A.q_spec += o; A.v_set += o; if (A.vm0) { A.vm0 += o; A.va0 += o; }
    A.vm += o; A.va += o; A.iterations += b0; A.converged += b0; if (A.final_norm) A.final_norm += b0;
    A.pivot = ctx_pivot(c) + b0; A.status = ctx_status(c) + b0; A.it = ctx_it(c) + b0; A.active = ctx_active(c);
    A.factors = c->factors + (size_t)g0 * G * c->fac_stride; A.work = c->work + (size_t)g0 * G * c->work_stride;
    A.trash_grp = ((c->opt.max_batch + G - 1) >> c->gsh) - g0;
    A.gsh = c->gsh; c->factor_gsh = c->gsh;
    if (c->opt.mode == SABLE_MODE_FUSED) {
        A.queue = c->ints + chunk;
        cudaError_t e = cudaMemsetAsync(A.queue, 0, 4, s);
        if (e != cudaSuccess) return e;
        A.t.level = c->level_fused;
        A.ring_r = c->ring_r; A.ring_slot = c->ring_slot; A.first_staged = c->first_staged;
        A.big_off = c->big_off; A.slot_off = c->slot_off; A.csz = c->csz; A.team_red = c->team_red + (size_t)chunk * c->grid * G;
        A.front_k = c->front_k; A.front_f0 = c->front_f0; A.front_level = c->front_level; A.front_off = c->front_off; A.front = c->front;
        // the attribute is per-function state shared by every live context: set it for THIS context right before the launch
        e = cudaFuncSetAttribute(fused_fn(sizeof(T) == 4, c->variant), cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem);
        if (e != cudaSuccess) return e;
        e = launch_fused<T>(c, A, s);
        c->launches += 1;
        return e;
    }
    // staged mode: one launch per stage; after three iterations the host reads the count of still-active scenarios after
    // every mismatch pass and stops launching when it is zero (this mode synchronises; it exists for per-stage profiling)
    A.t.level = c->level_stage;
    const int grid = (nb + G - 1) / G, th = c->threads_stage;
    if (c->opt.ir_sweeps > 0) {
        const size_t n = (size_t)c->opt.max_batch * c->T.n_bus;
        A.ir = 1; A.ir_v = reinterpret_cast<double2*>(c->irbuf) + o; A.ir_vm = c->irbuf + 2 * n + o;
        A.ir_dzp = c->irbuf + 3 * n + o; A.ir_dzq = c->irbuf + 4 * n + o; A.ir_bus_node = c->d_bus_node;
    }
    cudaError_t e = cudaMemsetAsync(A.active, 0, kMaxActive * 4, s);
    if (e != cudaSuccess) return e;
    k_st_init<T><<<grid, th, 0, s>>>(A);
    c->launches += 1;
    for (int i = 0; i <= A.max_it; ++i) {
        A.stage_it = std::min(i, kMaxActive - 1);
        if (i >= kMaxActive - 1) cudaMemsetAsync(A.active + A.stage_it, 0, 4, s);
        launch_st_mismatch_fill<T>(A, grid, th, s);
        c->launches += 1;
        if (i >= 3 || i == A.max_it) {
            int32_t left = 0;
            e = cudaMemcpyAsync(&left, A.active + A.stage_it, 4, cudaMemcpyDeviceToHost, s);
            if (e == cudaSuccess) e = cudaStreamSynchronize(s);
            if (e != cudaSuccess) return e;
            if (left == 0) break;
        }
        if (i == A.max_it) break;
        launch_st_factor_solve<T>(A, grid, th, s);
        c->launches += 1;
        if (!A.ir) continue;
        // inner refinement (ir_sweeps): dz from the FP32 factors, then `ir_sweeps` times r = -F1 - J1 dz in FP64, J1 c = r on the
        // same factors, dz += c in FP64; then the update.  Arrays of irbuf: 0-1 V, 2 |V|, 3-4 dz, 5-6 r, 7-8 c
        const size_t n = (size_t)c->opt.max_batch * c->T.n_bus, tot = (size_t)nb * c->T.n_bus;
        const int fb = (int)std::min<size_t>((tot + 255) / 256, 8192);
        k_st_ir_export<T><<<grid, th, 0, s>>>(A);
        IrArgs R{};
        R.n_bus = c->T.n_bus; R.batch = nb; R.fptr = c->fptr; R.fcol = c->fcol; R.fgb = c->fgb; R.bus_type = c->d_bus_type;
        R.status = A.status; R.p_spec = A.p_spec; R.q_spec = A.q_spec; R.v = A.ir_v; R.vm = A.ir_vm; R.dzp = A.ir_dzp; R.dzq = A.ir_dzq;
        R.rp = c->irbuf + 5 * n + o; R.rq = c->irbuf + 6 * n + o; R.long_rows = c->d_long; R.n_long = c->n_long;
        for (int sw = 0; sw < c->opt.ir_sweeps; ++sw) {
            k_ir_residual<<<fb, 256, 0, s>>>(R);
            if (launch_lin(c, b0, nb, c->irbuf + 5 * n, c->irbuf + 6 * n, 0, c->irbuf + 7 * n, c->irbuf + 8 * n, false, s) != SABLE_OK)
                return cudaErrorLaunchFailure;
            k_add2<<<fb, 256, 0, s>>>(A.ir_dzp, A.ir_dzq, c->irbuf + 7 * n + o, c->irbuf + 8 * n + o, tot);
            c->launches += 2;
        }
        k_st_ir_update<T><<<grid, th, 0, s>>>(A);
        c->launches += 2;
    }
    return cudaGetLastError();
}

static sable_status check_solve_args(sable_ctx* ctx, int32_t batch, const void* p_spec, const void* q_spec, const void* v_set,
                                     const void* vm0, const void* va0, double tol, int32_t max_it, const void* vm, const void* va,
                                     const void* iterations, const void* converged) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 0 || batch > ctx->opt.max_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch out of range");
    if (max_it < 0 || !(tol >= 0.0)) return fail(ctx, SABLE_ERR_INVALID_ARG, "max_it < 0 or tol < 0");
    if (batch > 0 && (!p_spec || !q_spec || !v_set || !vm || !va || !iterations || !converged || ((vm0 == nullptr) != (va0 == nullptr))))
        return fail(ctx, SABLE_ERR_INVALID_ARG, "null array (vm0 and va0 must both be given or both be NULL)");
    return SABLE_OK;
}

static SolveArgs base_args(sable_ctx* ctx, const double* p_spec, const double* q_spec, const double* v_set, const double* vm0,
                           const double* va0, double tol, int32_t max_it, double* vm, double* va, int32_t* iterations,
                           uint8_t* converged, double* final_norm) {
    SolveArgs A{};
    A.t = ctx->d; A.max_it = max_it; A.keep = ctx->opt.keep_factors; A.tol = tol;
    A.p_spec = p_spec; A.q_spec = q_spec; A.v_set = v_set; A.vm0 = vm0; A.va0 = va0;
    A.vm = vm; A.va = va; A.final_norm = final_norm; A.iterations = iterations; A.converged = converged;
    A.fac_stride = ctx->fac_stride; A.work_stride = ctx->work_stride; A.tim = ctx->tim;
    return A;
}

extern "C" sable_status sable_solve(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                    const double* v_set, const double* vm0, const double* va0, double tol, int32_t max_it,
                                    double* vm, double* va, int32_t* iterations, uint8_t* converged, double* final_norm,
                                    void* cuda_stream) {
    sable_status st = check_solve_args(ctx, batch, p_spec, q_spec, v_set, vm0, va0, tol, max_it, vm, va, iterations, converged);
    if (st != SABLE_OK) return st;
    ctx->have_factors = false; ctx->last_batch = batch;
    if (batch == 0) return SABLE_OK;                       /* empty batch: nothing is read or written */
    ON_DEVICE(ctx);
    const SolveArgs A = base_args(ctx, p_spec, q_spec, v_set, vm0, va0, tol, max_it, vm, va, iterations, converged, final_norm);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    CU(ctx->opt.precision == SABLE_MIXED ? launch_solve<float>(ctx, A, 0, batch, 0, s) : launch_solve<double>(ctx, A, 0, batch, 0, s));
    ctx->have_factors = ctx->opt.keep_factors != 0;
    return SABLE_OK;
}

extern "C" sable_status sable_get_pivot_flags(sable_ctx* ctx, int32_t batch, int32_t* flags, void* cuda_stream) {
    if (!ctx || !flags) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch != ctx->last_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch differs from the last sable_solve");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    CU(cudaMemcpyAsync(flags, ctx_pivot(ctx), (size_t)batch * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)cuda_stream));
    return SABLE_OK;
}

// ---- adjoint / linear solves on kept factors ---------------------------------------------------------------------
static sable_status launch_lin(sable_ctx* ctx, int b0, int batch, const double* rp, const double* rq, int transposed, double* xp,
                               double* xq, bool use_flags, cudaStream_t s) {
    LinArgs L{};
    const int gsh = ctx->factor_gsh, G = 1 << gsh, g0 = b0 >> gsh;
    const size_t o = (size_t)b0 * ctx->T.n_bus;
    L.t = ctx->d;
    L.t.level = gsh == 0 && gsh != ctx->gsh ? ctx->level_one : ctx->level_lin;
    L.batch = batch; L.transposed = transposed; L.gsh = gsh; L.rhs_p = rp + o; L.rhs_q = rq + o; L.x_p = xp + o; L.x_q = xq + o;
    L.pivot = use_flags ? ctx_pivot(ctx) + b0 : nullptr;
    L.factors = ctx->factors + (size_t)g0 * G * ctx->fac_stride; L.fac_stride = ctx->fac_stride;
    L.work = ctx->work + (size_t)g0 * G * ctx->work_stride; L.work_stride = ctx->work_stride;
    // the adjoint kernel follows the layout of the kernel that wrote the factors; with teams (cluster) when the NR kernel used them
    const int csz = gsh == ctx->gsh ? ctx->csz_lin : 1;
    const int th = gsh == 0 && gsh != ctx->gsh ? ctx->threads1 : ctx->threads_lin, grid = (batch + G - 1) / G * csz;
    L.big_off = (int)align16(big_bytes(th, gsh));
    L.csz = csz;
    const size_t rhs = ((size_t)ctx->T.n_node * 16) << gsh;
    int max_optin = 0; CU(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->opt.device));
    L.rhs_in_smem = csz == 1 && L.big_off + rhs <= std::min<size_t>((size_t)max_optin, 64 * 1024);
    size_t sm = L.big_off + (L.rhs_in_smem ? rhs : 0);
    // dense top front of the transposed sweeps: the NR kernel's front (same nodes, same assembly lists), when the factors were
    // written in this context's layout by a CTA working alone and the front still fits beside the right-hand sides
    if (transposed && csz == 1 && gsh == ctx->gsh && ctx->lin_front.k > 0) {
        const FrontPlan_& fp = ctx->lin_front;
        const size_t fb = (size_t)(ctx->opt.precision == SABLE_MIXED ? front_bytes<float>(fp.k, gsh) : front_bytes<double>(fp.k, gsh));
        if (align16(sm) + fb <= (size_t)max_optin) {
            L.front_k = fp.k; L.front_f0 = fp.f0; L.front_level = fp.level; L.front = fp.d;
            L.front_off = align16(sm); sm = L.front_off + fb;
        }
    }
    const void* lin = ctx->opt.precision == SABLE_MIXED ? (const void*)k_linsolve<float> : (const void*)k_linsolve<double>;
    CU(cudaFuncSetAttribute(lin, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max<size_t>(sm, 48 * 1024)));
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(th); cfg.dynamicSmemBytes = sm; cfg.stream = s;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = csz; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = csz > 1 ? 1 : 0;
    if (ctx->opt.precision == SABLE_MIXED) CU(cudaLaunchKernelEx(&cfg, k_linsolve<float>, L));
    else CU(cudaLaunchKernelEx(&cfg, k_linsolve<double>, L));
    ctx->launches += 1;
    return SABLE_OK;
}

extern "C" sable_status sable_adjoint(sable_ctx* ctx, int32_t batch, const double* g_va, const double* g_vm, double* lam_p,
                                      double* lam_q, void* cuda_stream) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (!ctx->have_factors) return fail(ctx, SABLE_ERR_STATE, "no kept factors: call sable_solve with keep_factors = 1 first");
    if (batch != ctx->last_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch differs from the last sable_solve");
    if (!g_va || !g_vm || !lam_p || !lam_q) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    return launch_lin(ctx, 0, batch, g_va, g_vm, 1, lam_p, lam_q, true, (cudaStream_t)cuda_stream);
}

// ---- Step-2 explicit recovery ---------------------------------------------------------------------------------------
extern "C" sable_status sable_recover(sable_ctx* ctx, int32_t batch, const double* vm, const double* va, double* p_inj,
                                      double* q_inj, void* cuda_stream) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 0 || batch > ctx->opt.max_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch out of range");
    if (batch == 0) return SABLE_OK;
    if (!vm || !va || !p_inj || !q_inj) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    ON_DEVICE(ctx);
    RecoverArgs R{};
    R.n_bus = ctx->T.n_bus; R.batch = batch; R.fptr = ctx->fptr; R.fcol = ctx->fcol; R.fgb = ctx->fgb;
    R.vm = vm; R.va = va; R.p_inj = p_inj; R.q_inj = q_inj; R.work = ctx->work; R.work_stride = ctx->work_stride;
    R.long_rows = ctx->d_long; R.n_long = ctx->n_long;
    const size_t sm = (size_t)ctx->T.n_bus * 16;
    R.v_in_smem = sm <= 160 * 1024;            // else the scenario's workspace slice (>= 3 (n_bus) 16 bytes) holds V
    if (ctx->placement == 2 && sm > 64 * 1024 && (size_t)batch * ctx->T.n_bus >= ((size_t)1 << 18)) {
        // large grids (V would take most of an SM's shared memory) with an HBM workspace: two launches over all (scenario, bus) pairs
        const int grid = (int)std::min<size_t>(((size_t)batch * ctx->T.n_bus + 255) / 256, 148 * 32);
        k_recover_flat<0><<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(R);
        k_recover_flat<1><<<grid, 256, 0, (cudaStream_t)cuda_stream>>>(R);
        ctx->launches += 2;
        CU(cudaGetLastError());
        return SABLE_OK;
    }
    if (R.v_in_smem && sm > 48 * 1024) CU(cudaFuncSetAttribute((const void*)k_recover, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int th = bus_threads(ctx->T.n_bus);
    k_recover<<<batch, th, R.v_in_smem ? sm : 0, (cudaStream_t)cuda_stream>>>(R);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return SABLE_OK;
}

// scratch of the layer / refinement calls: four [max_batch][n_bus] arrays, allocated at the first such call
static sable_status need_lbuf(sable_ctx* ctx) {
    if (ctx->lbuf) return SABLE_OK;
    void* p = nullptr;
    CU(cudaMalloc(&p, 4 * (size_t)ctx->opt.max_batch * ctx->T.n_bus * 8));
    ctx->dev_allocs.push_back(p); ctx->lbuf = (double*)p;
    return SABLE_OK;
}

// k_layer: a CTA per scenario, scratch in shared memory or (grids too large for that) in the scenario's workspace slice
static cudaError_t launch_layer(sable_ctx* ctx, LayerArgs& L, int batch, cudaStream_t s) {
    const size_t sm = (size_t)ctx->T.n_bus * 48;       // V, (P, Q), row weights
    L.in_smem = sm <= 160 * 1024;
    L.long_rows = ctx->d_long; L.n_long = ctx->n_long;
    if (L.in_smem && sm > 48 * 1024) { cudaError_t e = cudaFuncSetAttribute((const void*)k_layer, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm); if (e != cudaSuccess) return e; }
    k_layer<<<batch, bus_threads(ctx->T.n_bus), L.in_smem ? sm : 0, s>>>(L);
    ctx->launches += 1;
    return cudaGetLastError();
}

// ---- implicit-layer backward ----------------------------------------------------------------------------------------
extern "C" sable_status sable_layer_backward(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                             const double* gl_pg, const double* gl_qg, const double* gl_vm, const double* gl_va,
                                             double* dx_pg, double* dx_vm, void* cuda_stream) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (!ctx->have_factors) return fail(ctx, SABLE_ERR_STATE, "no kept factors: call sable_solve with keep_factors = 1 first");
    if (batch != ctx->last_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch differs from the last sable_solve");
    if (!vm || !va || !gl_pg || !gl_qg || !gl_vm || !gl_va || !dx_pg || !dx_vm) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    sable_status st = need_lbuf(ctx); if (st != SABLE_OK) return st;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)ctx->opt.max_batch * ctx->T.n_bus;
    LayerArgs L{};
    L.n_bus = ctx->T.n_bus; L.batch = batch; L.fptr = ctx->fptr; L.fcol = ctx->fcol; L.ftpos = ctx->ftpos; L.fgb = ctx->fgb;
    L.bus_type = ctx->d_bus_type; L.vm = vm; L.va = va; L.gl_pg = gl_pg; L.gl_qg = gl_qg; L.gl_vm = gl_vm; L.gl_va = gl_va;
    L.g_va = ctx->lbuf; L.g_vm = ctx->lbuf + n; L.lam_p = ctx->lbuf + 2 * n; L.lam_q = ctx->lbuf + 3 * n;
    L.dx_pg = dx_pg; L.dx_vm = dx_vm; L.work = ctx->work; L.work_stride = ctx->work_stride;
    L.post = 0;
    CU(launch_layer(ctx, L, batch, s));
    st = launch_lin(ctx, 0, batch, L.g_va, L.g_vm, 1, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, true, s);
    if (st != SABLE_OK) return st;
    L.post = 1;
    CU(launch_layer(ctx, L, batch, s));
    return SABLE_OK;
}

// ---- adjoint with FP64 iterative refinement -------------------------------------------------------------------------
extern "C" sable_status sable_adjoint_refined(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                              const double* g_va, const double* g_vm, int32_t sweeps, double* lam_p,
                                              double* lam_q, void* cuda_stream) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (!ctx->have_factors) return fail(ctx, SABLE_ERR_STATE, "no kept factors: call sable_solve with keep_factors = 1 first");
    if (batch != ctx->last_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch differs from the last sable_solve");
    if (!vm || !va || !g_va || !g_vm || !lam_p || !lam_q) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    if (sweeps < 0 || sweeps > 16) return fail(ctx, SABLE_ERR_INVALID_ARG, "sweeps out of range [0, 16]");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    cudaStream_t s = (cudaStream_t)cuda_stream;
    sable_status st = launch_lin(ctx, 0, batch, g_va, g_vm, 1, lam_p, lam_q, true, s);
    if (st != SABLE_OK || sweeps == 0) return st;
    st = need_lbuf(ctx); if (st != SABLE_OK) return st;
    const size_t n = (size_t)ctx->opt.max_batch * ctx->T.n_bus, nb = (size_t)batch * ctx->T.n_bus;
    LayerArgs L{};
    L.n_bus = ctx->T.n_bus; L.batch = batch; L.fptr = ctx->fptr; L.fcol = ctx->fcol; L.ftpos = ctx->ftpos; L.fgb = ctx->fgb;
    L.bus_type = ctx->d_bus_type; L.vm = vm; L.va = va; L.gl_va = g_va; L.gl_vm = g_vm; L.lam_p = lam_p; L.lam_q = lam_q;
    L.g_va = ctx->lbuf; L.g_vm = ctx->lbuf + n; L.work = ctx->work; L.work_stride = ctx->work_stride; L.post = 2;
    for (int it = 0; it < sweeps; ++it) {
        CU(launch_layer(ctx, L, batch, s));                                                 // r = g - J1^T lambda   (FP64)
        st = launch_lin(ctx, 0, batch, L.g_va, L.g_vm, 1, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, false, s);   // J1^T d = r  (kept factors)
        if (st != SABLE_OK) return st;
        k_add2<<<(int)std::min<size_t>((nb + 255) / 256, 4096), 256, 0, s>>>(lam_p, lam_q, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, nb);
        CU(cudaGetLastError());
        ctx->launches += 1;
    }
    return SABLE_OK;
}

// ---- host-buffer wrappers (end-to-end path: H2D, solve, D2H; synchronous) ------------------------------------------
// The batch is cut into up to kMaxChunk chunks of whole groups, each on its own stream: copy in, kernel, copy out.  The
// copies of one chunk overlap the kernels of the others (and the kernels one another: every chunk has its own queue
// counter and its own part of the workspace), so the exposed copy time is about that of one chunk.
static sable_status need_hbuf(sable_ctx* ctx) {
    if (ctx->hbuf) return SABLE_OK;
    const size_t mb = (size_t)ctx->opt.max_batch, nb = (size_t)ctx->T.n_bus;
    void *a = nullptr, *b = nullptr, *c = nullptr;
    CU(cudaMalloc(&a, 9 * mb * nb * 8 + mb * 8)); ctx->dev_allocs.push_back(a); ctx->hbuf = (double*)a;
    CU(cudaMalloc(&b, mb * 4)); ctx->dev_allocs.push_back(b); ctx->hbuf_it = (int32_t*)b;
    CU(cudaMalloc(&c, mb)); ctx->dev_allocs.push_back(c); ctx->hbuf_cv = (uint8_t*)c;
    for (int i = 0; i < kMaxChunk; ++i) CU(cudaStreamCreateWithFlags(&ctx->hstream[i], cudaStreamNonBlocking));
    return SABLE_OK;
}
static int host_chunks(const sable_ctx* ctx, int batch, int* per) {
    const int G = 1 << ctx->gsh, groups = (batch + G - 1) / G;
    // a chunk should still give every SM its CTAs; a staged-mode solve synchronises inside, so it is not cut
    int n = ctx->opt.mode == SABLE_MODE_STAGED ? 1 : std::max(1, std::min(kMaxChunk, groups / std::max(1, ctx->grid / 4)));
    n = std::max(1, std::min(n, groups));
    *per = (groups + n - 1) / n * G;
    return (batch + *per - 1) / *per;
}

extern "C" sable_status sable_solve_host(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                         const double* v_set, const double* vm0, const double* va0, double tol,
                                         int32_t max_it, double* vm, double* va, int32_t* iterations, uint8_t* converged,
                                         double* final_norm) {
    sable_status st = check_solve_args(ctx, batch, p_spec, q_spec, v_set, vm0, va0, tol, max_it, vm, va, iterations, converged);
    if (st != SABLE_OK) return st;
    ctx->have_factors = false; ctx->last_batch = batch;
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    st = need_hbuf(ctx); if (st != SABLE_OK) return st;
    const size_t nbus = (size_t)ctx->T.n_bus, n = (size_t)ctx->opt.max_batch * nbus;
    double* d = ctx->hbuf;       // slots: 0 p, 1 q, 2 vset, 3 vm0, 4 va0, 5 vm, 6 va, (7, 8 adjoint), then norm
    double* dn = ctx->hbuf + 9 * n;
    const SolveArgs A = base_args(ctx, d, d + n, d + 2 * n, vm0 ? d + 3 * n : nullptr, vm0 ? d + 4 * n : nullptr, tol, max_it,
                                  d + 5 * n, d + 6 * n, ctx->hbuf_it, ctx->hbuf_cv, dn);
    int per = 0;
    const int nch = host_chunks(ctx, batch, &per);
    for (int c = 0; c < nch; ++c) {
        const int b0 = c * per, nb = std::min(per, batch - b0);
        const size_t o = (size_t)b0 * nbus, bytes = (size_t)nb * nbus * 8;
        cudaStream_t s = ctx->hstream[c];
        CU(cudaMemcpyAsync(d + o, p_spec + o, bytes, cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(d + n + o, q_spec + o, bytes, cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(d + 2 * n + o, v_set + o, bytes, cudaMemcpyHostToDevice, s));
        if (vm0) { CU(cudaMemcpyAsync(d + 3 * n + o, vm0 + o, bytes, cudaMemcpyHostToDevice, s)); CU(cudaMemcpyAsync(d + 4 * n + o, va0 + o, bytes, cudaMemcpyHostToDevice, s)); }
        CU(ctx->opt.precision == SABLE_MIXED ? launch_solve<float>(ctx, A, b0, nb, c, s) : launch_solve<double>(ctx, A, b0, nb, c, s));
        CU(cudaMemcpyAsync(vm + o, d + 5 * n + o, bytes, cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(va + o, d + 6 * n + o, bytes, cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(iterations + b0, ctx->hbuf_it + b0, (size_t)nb * 4, cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(converged + b0, ctx->hbuf_cv + b0, (size_t)nb, cudaMemcpyDeviceToHost, s));
        if (final_norm) CU(cudaMemcpyAsync(final_norm + b0, dn + b0, (size_t)nb * 8, cudaMemcpyDeviceToHost, s));
    }
    for (int c = 0; c < nch; ++c) CU(cudaStreamSynchronize(ctx->hstream[c]));
    ctx->have_factors = ctx->opt.keep_factors != 0;
    return SABLE_OK;
}

extern "C" sable_status sable_adjoint_host(sable_ctx* ctx, int32_t batch, const double* g_va, const double* g_vm,
                                           double* lam_p, double* lam_q) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (!ctx->have_factors) return fail(ctx, SABLE_ERR_STATE, "no kept factors: call sable_solve_host with keep_factors = 1 first");
    if (batch != ctx->last_batch || !g_va || !g_vm || !lam_p || !lam_q) return fail(ctx, SABLE_ERR_INVALID_ARG, "bad argument");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    sable_status st = need_hbuf(ctx); if (st != SABLE_OK) return st;
    const size_t nbus = (size_t)ctx->T.n_bus, n = (size_t)ctx->opt.max_batch * nbus;
    double* d = ctx->hbuf;
    int per = 0;
    const int nch = host_chunks(ctx, batch, &per);
    for (int c = 0; c < nch; ++c) {
        const int b0 = c * per, nb = std::min(per, batch - b0);
        const size_t o = (size_t)b0 * nbus, bytes = (size_t)nb * nbus * 8;
        cudaStream_t s = ctx->hstream[c];
        CU(cudaMemcpyAsync(d + o, g_va + o, bytes, cudaMemcpyHostToDevice, s));
        CU(cudaMemcpyAsync(d + n + o, g_vm + o, bytes, cudaMemcpyHostToDevice, s));
        st = launch_lin(ctx, b0, nb, d, d + n, 1, d + 7 * n, d + 8 * n, true, s);
        if (st != SABLE_OK) return st;
        CU(cudaMemcpyAsync(lam_p + o, d + 7 * n + o, bytes, cudaMemcpyDeviceToHost, s));
        CU(cudaMemcpyAsync(lam_q + o, d + 8 * n + o, bytes, cudaMemcpyDeviceToHost, s));
    }
    for (int c = 0; c < nch; ++c) CU(cudaStreamSynchronize(ctx->hstream[c]));
    return SABLE_OK;
}

// ---- per-stage times in the default workspace layout (debug / measurement) ------------------------------------------------
// Runs the staged kernels (the fused kernel's own stage routines, one stage per launch, group-interleaved workspace) for
// three Newton iterations from the flat start on the given batch and returns the mean CUDA-event time of the mismatch +
// fill launch and of the refactor + solve launch (ms) -- all scenarios are still active in those iterations.  Synchronous;
// overwrites the workspace (kept factors are gone).
extern "C" sable_status sable_debug_stage_times(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                                const double* v_set, double* ms_mismatch_fill, double* ms_factor_solve, void* cuda_stream) {
    if (!ctx || !ms_mismatch_fill || !ms_factor_solve) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 1 || batch > ctx->opt.max_batch || !p_spec || !q_spec || !v_set) return fail(ctx, SABLE_ERR_INVALID_ARG, "bad argument");
    ON_DEVICE(ctx);
    sable_status st = need_lbuf(ctx); if (st != SABLE_OK) return st;     // outputs nobody reads: vm, va -> lbuf
    ctx->have_factors = false;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)ctx->opt.max_batch * ctx->T.n_bus;
    SolveArgs A = base_args(ctx, p_spec, q_spec, v_set, nullptr, nullptr, 0.0, 1000, ctx->lbuf, ctx->lbuf + n, ctx_it(ctx), (uint8_t*)(ctx->lbuf + 2 * n), nullptr);
    A.iterations = (int32_t*)(ctx->lbuf + 3 * n);
    A.keep = 0; A.batch = batch;
    A.pivot = ctx_pivot(ctx); A.status = ctx_status(ctx); A.it = ctx_it(ctx); A.active = ctx_active(ctx); A.stage_it = 0;
    A.factors = ctx->factors; A.work = ctx->work;
    const int G = 1 << ctx->gsh;
    A.trash_grp = (ctx->opt.max_batch + G - 1) >> ctx->gsh; A.gsh = ctx->gsh; ctx->factor_gsh = ctx->gsh;
    A.t.level = ctx->level_stage;
    const int grid = (batch + G - 1) / G, th = ctx->threads_stage;
    const bool mixed = ctx->opt.precision == SABLE_MIXED;
    cudaEvent_t ev[7];
    for (auto& e : ev) CU(cudaEventCreate(&e));
    if (mixed) k_st_init<float><<<grid, th, 0, s>>>(A); else k_st_init<double><<<grid, th, 0, s>>>(A);
    for (int i = 0; i < 3; ++i) {
        CU(cudaEventRecord(ev[2 * i], s));
        if (mixed) launch_st_mismatch_fill<float>(A, grid, th, s); else launch_st_mismatch_fill<double>(A, grid, th, s);
        CU(cudaEventRecord(ev[2 * i + 1], s));
        if (mixed) launch_st_factor_solve<float>(A, grid, th, s); else launch_st_factor_solve<double>(A, grid, th, s);
    }
    CU(cudaEventRecord(ev[6], s));
    CU(cudaStreamSynchronize(s));
    CU(cudaGetLastError());
    ctx->launches += 7;
    double a = 0, b = 0;
    for (int i = 0; i < 3; ++i) {
        float x = 0, y = 0;
        CU(cudaEventElapsedTime(&x, ev[2 * i], ev[2 * i + 1]));
        CU(cudaEventElapsedTime(&y, ev[2 * i + 1], ev[2 * i + 2]));
        a += x / 3.0; b += y / 3.0;
    }
    for (auto& e : ev) cudaEventDestroy(e);
    *ms_mismatch_fill = a; *ms_factor_solve = b;
    return SABLE_OK;
}

extern "C" sable_status sable_debug_timing(sable_ctx* ctx, uint64_t* out, int32_t n) {
    if (!ctx || !out) return SABLE_ERR_INVALID_ARG;
    if (!ctx->tim) return fail(ctx, SABLE_ERR_STATE, "timing counters are off (create the context with SABLE_TIMING=1 in the environment)");
    const int have = 4 * ctx->T.n_level + 4;
    CU(cudaMemcpy(out, ctx->tim, (size_t)std::min(n, have) * 8, cudaMemcpyDeviceToHost));
    CU(cudaMemset(ctx->tim, 0, (size_t)have * 8));
    return SABLE_OK;
}

// ---- debug exports -----------------------------------------------------------------------------------------------
extern "C" sable_status sable_debug_pattern(const sable_ctx* c, int32_t* node_bus, int32_t* node_level, int32_t* pair_ptr,
                                            int32_t* pair_col, uint8_t* pair_in_j, int32_t* term_ptr, int32_t* term_a,
                                            int32_t* term_b, int32_t* dterm_ptr, int32_t* dterm) {
    if (!c) return SABLE_ERR_INVALID_ARG;
    const Template& T = c->T;
    auto cp = [](auto* dst, const auto& v) { if (dst && !v.empty()) memcpy(dst, v.data(), v.size() * sizeof(v[0])); };
    cp(node_bus, T.node_bus); cp(node_level, T.node_level); cp(pair_ptr, T.pair_ptr); cp(pair_col, T.pair_col);
    cp(term_ptr, T.term_ptr); cp(term_a, T.term_a); cp(term_b, T.term_b); cp(dterm_ptr, T.dterm_ptr); cp(dterm, T.dterm);
    if (pair_in_j) for (size_t p = 0; p < T.pair_yu.size(); ++p) pair_in_j[p] = T.pair_yu[p] >= 0;
    return SABLE_OK;
}

static sable_status launch_debug(sable_ctx* ctx, DebugArgs& D, cudaStream_t s) {
    D.t = ctx->d; D.t.level = ctx->level_one; D.zeros = ctx->zeros; ctx->factor_gsh = 0; D.pivot = D.what == 2 ? ctx_pivot(ctx) : nullptr;
    D.factors = ctx->factors; D.work = ctx->work; D.fac_stride = ctx->fac_stride; D.work_stride = ctx->work_stride;
    if (ctx->opt.precision == SABLE_MIXED) k_debug<float><<<D.batch, ctx->threads1, 0, s>>>(D);
    else k_debug<double><<<D.batch, ctx->threads1, 0, s>>>(D);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return SABLE_OK;
}
static sable_status debug_check(sable_ctx* ctx, int batch) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 1 || batch > ctx->opt.max_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch out of range");
    ctx->have_factors = false; ctx->last_batch = batch;
    return SABLE_OK;
}

extern "C" sable_status sable_debug_mismatch(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                             const double* vm, const double* va, double* f_p, double* f_q, double* norm,
                                             void* cuda_stream) {
    sable_status st = debug_check(ctx, batch); if (st) return st;
    ON_DEVICE(ctx);
    if (!p_spec || !q_spec || !vm || !va || !f_p || !f_q || !norm) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    DebugArgs D{}; D.batch = batch; D.what = 0; D.p_spec = p_spec; D.q_spec = q_spec; D.vm = vm; D.va = va; D.f_p = f_p; D.f_q = f_q; D.norm = norm;
    return launch_debug(ctx, D, (cudaStream_t)cuda_stream);
}

extern "C" sable_status sable_debug_jacobian(sable_ctx* ctx, int32_t batch, const double* vm, const double* va, double* diag,
                                             double* pairs, void* cuda_stream) {
    sable_status st = debug_check(ctx, batch); if (st) return st;
    ON_DEVICE(ctx);
    if (!vm || !va || !diag || !pairs) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    DebugArgs D{}; D.batch = batch; D.what = 1; D.vm = vm; D.va = va; D.diag = diag; D.pairs = pairs;
    return launch_debug(ctx, D, (cudaStream_t)cuda_stream);
}

extern "C" sable_status sable_debug_linear_solve(sable_ctx* ctx, int32_t batch, const double* vm, const double* va,
                                                 const double* rhs_p, const double* rhs_q, int32_t transpose, double* x_p,
                                                 double* x_q, void* cuda_stream) {
    sable_status st = debug_check(ctx, batch); if (st) return st;
    ON_DEVICE(ctx);
    if (!vm || !va || !rhs_p || !rhs_q || !x_p || !x_q) return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    DebugArgs D{}; D.batch = batch; D.what = 2; D.vm = vm; D.va = va;
    st = launch_debug(ctx, D, (cudaStream_t)cuda_stream); if (st) return st;
    return launch_lin(ctx, 0, batch, rhs_p, rhs_q, transpose ? 1 : 0, x_p, x_q, false, (cudaStream_t)cuda_stream);
}
