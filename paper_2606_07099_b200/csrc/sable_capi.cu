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

struct sable_ctx {
    Template T;
    sable_options opt{};
    sable_info info{};
    DevTemplate d{};
    std::vector<void*> dev_allocs;
    char* factors = nullptr;  char* work = nullptr;  int32_t* ints = nullptr;   // ints: queue[1] status[mb] it[mb]
    double* zeros = nullptr;
    const int32_t* fptr = nullptr; const int32_t* fcol = nullptr; const double2* fgb = nullptr;   // full Y_bus, bus order
    const int32_t* ftpos = nullptr; const uint8_t* d_bus_type = nullptr; double* lbuf = nullptr;   // layer backward
    unsigned long long* tim = nullptr;                       // SABLE_TIMING=1: per-phase cycle counters of CTA 0
    int64_t fac_stride = 0, work_stride = 0;                 // bytes per scenario
    // launch plan of the fused kernel (choose_launch) and of the one-scenario-per-CTA kernels
    int threads = 0, grid = 0, placement = 0, smem = 0, gsh = 0, ctas_per_sm = 1;
    int dg_cut = 0, pr_cut = 0, st_cut = 0, cut_level = 0;
    int threads1 = 0;                                        // staged / adjoint / debug kernels
    int factor_gsh = 0;                                      // group layout of the factors currently in the workspace
    const LevelDesc* level_fused = nullptr; const LevelDesc* level_one = nullptr; const LevelDesc* level_lin = nullptr;
    int threads_lin = 0;                                     // adjoint kernel on group-interleaved factors
    std::vector<LevelDesc> lv_host;                          // blob offsets per level (splits filled per kernel family)
    std::vector<char> blob_host;
    int ring_r = 0, ring_slot = 0, first_staged = 0;
    int front_k = 0, front_f0 = 0, front_level = 0; int64_t front_off = 0; LevelDesc front{};   // dense top front (sable_front.cuh)
    int last_batch = -1;  bool have_factors = false;
    int64_t launches = 0;
    std::string err;
    // host wrapper staging (device)
    double* hbuf = nullptr; int32_t* hbuf_it = nullptr; uint8_t* hbuf_cv = nullptr;
};

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
    I.ctas_per_sm = c->ctas_per_sm; I.slots_per_cta = 1 << c->gsh; I.cut_level = c->cut_level;
    I.front_k = c->front_k; I.front_level = c->front_k > 0 ? c->front_level : T.n_level;
}

// kernel variant: placement 0 = on chip, 1 = mixed (only on request: SABLE_CUT), 2 = HBM; small = up to 128 threads
static const void* fused_fn(bool mixed, int place, bool small) {
    if (place == 0) return mixed ? (const void*)k_nr_fused<float, 0, false> : (const void*)k_nr_fused<double, 0, false>;
    if (place == 1) return mixed ? (const void*)k_nr_fused<float, 1, false> : (const void*)k_nr_fused<double, 1, false>;
    if (small) return mixed ? (const void*)k_nr_fused<float, 2, true> : (const void*)k_nr_fused<double, 2, true>;
    return mixed ? (const void*)k_nr_fused<float, 2, false> : (const void*)k_nr_fused<double, 2, false>;
}

// threads per CTA of the one-thread-per-bus kernels (recover, layer): whole rounds with no idle tail (300 buses -> 160
// threads x 2 rounds, not 256 x 2 with the second round 85 % idle), 64 for small grids, 512 for large ones
static int bus_threads(int n_bus) {
    if (n_bus <= 256) return 64;
    const int cap = n_bus <= 4096 ? 256 : 512, rounds = (n_bus + cap - 1) / cap;
    return std::min(cap, ((n_bus + rounds - 1) / rounds + 31) / 32 * 32);
}

static int env_int(const char* name, int dflt) { const char* e = getenv(name); return e ? atoi(e) : dflt; }

// lanes per target (log2) for a level with n targets whose longest list has max_len entries: as many as keep every
// thread busy at most once, never more than a warp's share per slot
static uint8_t pick_split(int n, int max_len, int threads, int gsh) {
    int s = 0;
    while ((2 << s) <= (32 >> gsh) && (int64_t)n * (2 << s) <= (threads >> gsh) && (2 << s) <= std::max(1, max_len)) ++s;
    return (uint8_t)s;
}

// level slices of the index program (layout: LevelDesc in sable_device.cuh)
static void build_blobs(const Template& T, std::vector<LevelDesc>& lv, std::vector<char>& blob) {
    lv.assign(T.n_level, LevelDesc{});
    blob.clear();
    auto al = [](size_t x, size_t a) { return (x + a - 1) / a * a; };
    for (int l = 0; l < T.n_level; ++l) {
        LevelDesc& d = lv[l];
        d.m0 = T.level_ptr[l]; d.m1 = T.level_ptr[l + 1]; d.p0 = T.pair_ptr[d.m0]; d.p1 = T.pair_ptr[d.m1];
        const int nm = d.m1 - d.m0, np = d.p1 - d.p0;
        const int nd = T.dterm_ptr[d.m1] - T.dterm_ptr[d.m0], nt = T.term_ptr[d.p1] - T.term_ptr[d.p0];
        size_t o = 0;
        o += (size_t)(nm + 1) * 4; d.o_tptr = (int32_t)o;
        o += (size_t)(np + 1) * 4; d.o_pptr = (int32_t)o;
        o += (size_t)(nm + 1) * 4; o = al(o, 8); d.o_dak = (int32_t)o;
        o += (size_t)nd * 8; d.o_pmj = (int32_t)o;
        o += (size_t)np * 8; d.o_tab = (int32_t)o;
        o += (size_t)nt * 8; d.o_py = (int32_t)o;              // (the Y values of the pairs live in DevTemplate::pair_y)
        o = al(o, 128);
        d.blob_off = (int32_t)blob.size(); d.blob_bytes = (int32_t)o;
        blob.resize(blob.size() + o, 0);
        char* base = blob.data() + d.blob_off;
        int32_t* dptr = (int32_t*)base; int32_t* tptr = (int32_t*)(base + d.o_tptr); int32_t* pptr = (int32_t*)(base + d.o_pptr);
        int2* dak = (int2*)(base + d.o_dak); int2* pmj = (int2*)(base + d.o_pmj); int2* tab = (int2*)(base + d.o_tab);
        for (int i = 0; i <= nm; ++i) {
            dptr[i] = T.dterm_ptr[d.m0 + i] - T.dterm_ptr[d.m0];
            pptr[i] = (T.pair_ptr[d.m0 + i] - d.p0) | ((i < nm && T.node_pq[d.m0 + i]) ? 1 << 30 : 0);
        }
        for (int i = 0; i <= np; ++i) tptr[i] = T.term_ptr[d.p0 + i] - T.term_ptr[d.p0];
        for (int q = 0; q < nd; ++q) { const int a = T.dterm[T.dterm_ptr[d.m0] + q]; dak[q] = make_int2(a, T.pair_row[a]); }
        for (int q = 0; q < nt; ++q) tab[q] = make_int2(T.term_a[T.term_ptr[d.p0] + q], T.term_b[T.term_ptr[d.p0] + q]);
        for (int i = 0; i < np; ++i) {
            const int p = d.p0 + i, m = T.pair_row[p], j = T.pair_col[p];
            pmj[i] = make_int2(m | (T.node_pq[m] ? 1 << 30 : 0), j | (T.node_pq[j] ? 1 << 30 : 0));
        }
    }
}

// lane splits for a kernel family (threads per CTA, slots per CTA) and the streamed-level flag
static std::vector<LevelDesc> build_levels(const Template& T, const std::vector<LevelDesc>& base, int threads, int gsh, int first_staged) {
    std::vector<LevelDesc> lv(base);
    for (int l = 0; l < T.n_level; ++l) {
        LevelDesc& d = lv[l];
        int maxd = 0, maxt = 0, maxb = 0;
        for (int m = d.m0; m < d.m1; ++m) {
            maxd = std::max(maxd, T.dterm_ptr[m + 1] - T.dterm_ptr[m]);
            maxb = std::max(maxb, T.pair_ptr[m + 1] - T.pair_ptr[m]);
        }
        for (int p = d.p0; p < d.p1; ++p) maxt = std::max(maxt, T.term_ptr[p + 1] - T.term_ptr[p]);
        d.sd = pick_split(d.m1 - d.m0, maxd, threads, gsh);
        d.sp = pick_split(d.p1 - d.p0, maxt, threads, gsh);
        d.sb = pick_split(d.m1 - d.m0, maxb, threads, gsh);
        d.staged = l >= first_staged;
    }
    return lv;
}

// Dense top front (sable_front.cuh): the nodes of the last elimination levels, as many levels as keep the K x K block
// matrix within `budget` bytes of shared memory per CTA (K <= kcap).  Appends the assembly lists (the front targets'
// multiply-subtract terms whose eliminated node k lies below the front) to the blob and fills ctx->front*.
static void build_front(sable_ctx* c, int threads, int gsh, int64_t budget, int kcap) {
    const Template& T = c->T;
    const int nn = T.n_node, np = (int)T.pair_col.size(), nl = T.n_level;
    const bool mixed = c->opt.precision == SABLE_MIXED;
    c->front_k = 0; c->front_f0 = nn; c->front_level = nl; c->front = LevelDesc{};
    auto bytes = [&](int K) { return mixed ? front_bytes<float>(K, gsh) : front_bytes<double>(K, gsh); };
    int lc = nl;
    while (lc > 1 && nn - T.level_ptr[lc - 1] <= kcap && bytes(nn - T.level_ptr[lc - 1]) <= budget) --lc;
    if (nl - lc < 2) return;                                 // merging fewer than two levels saves nothing
    const int f0 = T.level_ptr[lc], K = nn - f0;
    LevelDesc d{};
    d.m0 = f0; d.m1 = nn; d.p0 = T.pair_ptr[f0]; d.p1 = np;
    const int nm = K, npr = d.p1 - d.p0;
    std::vector<int32_t> dptr(nm + 1, 0), tptr(npr + 1, 0);
    std::vector<int2> dak, tab, pmj(npr);
    int maxd = 0, maxt = 0;
    for (int i = 0; i < nm; ++i) {
        for (int q = T.dterm_ptr[f0 + i]; q < T.dterm_ptr[f0 + i + 1]; ++q) {
            const int a = T.dterm[q], k = T.pair_row[a];
            if (k < f0) dak.push_back(make_int2(a, k));
        }
        dptr[i + 1] = (int32_t)dak.size(); maxd = std::max(maxd, dptr[i + 1] - dptr[i]);
    }
    for (int i = 0; i < npr; ++i) {
        const int p = d.p0 + i;
        for (int q = T.term_ptr[p]; q < T.term_ptr[p + 1]; ++q)
            if (T.pair_row[T.term_a[q]] < f0) tab.push_back(make_int2(T.term_a[q], T.term_b[q]));
        tptr[i + 1] = (int32_t)tab.size(); maxt = std::max(maxt, tptr[i + 1] - tptr[i]);
        const int m = T.pair_row[p], j = T.pair_col[p];
        pmj[i] = make_int2(m | (T.node_pq[m] ? 1 << 30 : 0), j | (T.node_pq[j] ? 1 << 30 : 0));
    }
    auto al = [](size_t x, size_t a) { return (x + a - 1) / a * a; };
    size_t o = 0;
    o += (size_t)(nm + 1) * 4; d.o_tptr = (int32_t)o;
    o += (size_t)(npr + 1) * 4; d.o_pptr = (int32_t)o; o = al(o, 8); d.o_dak = (int32_t)o;
    o += dak.size() * 8; d.o_pmj = (int32_t)o;
    o += (size_t)npr * 8; d.o_tab = (int32_t)o;
    o += tab.size() * 8; o = al(o, 128); d.o_py = (int32_t)o;
    d.blob_off = (int32_t)c->blob_host.size(); d.blob_bytes = (int32_t)o;
    c->blob_host.resize(c->blob_host.size() + o, 0);
    char* base = c->blob_host.data() + d.blob_off;
    memcpy(base, dptr.data(), dptr.size() * 4);
    memcpy(base + d.o_tptr, tptr.data(), tptr.size() * 4);
    if (!dak.empty()) memcpy(base + d.o_dak, dak.data(), dak.size() * 8);
    if (!pmj.empty()) memcpy(base + d.o_pmj, pmj.data(), pmj.size() * 8);
    if (!tab.empty()) memcpy(base + d.o_tab, tab.data(), tab.size() * 8);
    d.sd = pick_split(nm, maxd, threads, gsh);
    d.sp = pick_split(npr, maxt, threads, gsh);
    c->front = d; c->front_k = K; c->front_f0 = f0; c->front_level = lc;
}

// Launch plan of the fused kernel: as many scenario slots per CTA as fit entirely in shared
// memory (G = 8, 4, 2, 1); if not even one fits, one slot per CTA with the top of the elimination tree (levels >=
// cut_level) on chip and the wide early levels in the scenario's HBM slice.
static sable_status choose_launch(sable_ctx* ctx) {
    const Template& T = ctx->T;
    const int nn = T.n_node, np = (int)T.pair_col.size(), nl = T.n_level;
    const bool mixed = ctx->opt.precision == SABLE_MIXED;
    int dev = 0; CU(cudaGetDevice(&dev));
    int max_optin = 0, n_sm = 0, smem_sm = 0;
    CU(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    CU(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    CU(cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    int ring_bytes = 0;
    auto need = [&](int gsh, int dgc, int prc, int stc) {
        return mixed ? smem_need<float>(nn, np, nl, ring_bytes, gsh, dgc, prc, stc) : smem_need<double>(nn, np, nl, ring_bytes, gsh, dgc, prc, stc);
    };
    // ring candidates (slots, slot capacity): the streamed levels are the trailing run of levels whose blobs fit a slot
    struct RingOpt { int r, cap; };
    const int r_env = env_int("SABLE_RING_R", -1), cap_env = env_int("SABLE_RING_SLOT", -1);
    std::vector<RingOpt> ropts = {{3, 8192}, {2, 8192}, {3, 4096}, {2, 4096}, {2, 2048}, {0, 0}};
    if (r_env >= 0 || cap_env >= 0) ropts = {{r_env >= 0 ? r_env : 3, cap_env >= 0 ? cap_env : 8192}, {0, 0}};
    auto set_ring = [&](const RingOpt& o) {
        int first = nl, slot = 0;
        if (o.r > 0) while (first > 0 && ctx->lv_host[first - 1].blob_bytes <= o.cap) { --first; slot = std::max(slot, ctx->lv_host[first].blob_bytes); }
        if (first == nl) { ctx->ring_r = 0; ctx->ring_slot = 0; ctx->first_staged = nl; ring_bytes = 0; return; }
        ctx->ring_r = o.r; ctx->ring_slot = slot; ctx->first_staged = first; ring_bytes = o.r * slot;
    };
    int th = ctx->opt.threads;
    if (th <= 0) th = nn <= 64 ? 64 : nn <= 200 ? 256 : (nn > 1200 && nn <= 4000) ? 256 : 512;   // measured: profiles/r01_v2_sweeps.md
    th = env_int("SABLE_THREADS", th);
    th = std::min(512, std::max(32, (th + 31) / 32 * 32));
    const int mb = ctx->opt.max_batch;
    int gsh = -1, want_ctas = 1;
    const int g_env = env_int("SABLE_G", 0);
    for (int cand = 3; cand >= 0 && gsh < 0; --cand) {
        if (g_env > 0 && (1 << cand) != g_env) continue;
        // do not group more scenarios per CTA than leaves every SM a CTA (small batches stay spread out)
        if (g_env <= 0 && cand > 0 && (int64_t)n_sm * (1 << cand) > (int64_t)mb) continue;
        // the blob ring pays only where the slots leave no L1 for the index program (measured: cfg 2 with 57 KB of L1
        // left runs 0.133 ms without the ring, 0.147 ms with it; cfg 3 on chip with 21 KB left 4.9 ms vs 4.4 ms)
        if (r_env < 0 && cap_env < 0) {
            set_ring(RingOpt{0, 0});
            const int64_t n0 = need(cand, 0, 0, 0) + 1024;
            if (n0 <= max_optin && smem_sm - (smem_sm / n0) * n0 >= 32 * 1024) { gsh = cand; break; }
        }
        for (const RingOpt& o : ropts) {
            set_ring(o);
            if (need(cand, 0, 0, 0) <= max_optin) { gsh = cand; break; }
        }
    }
    const int cut_env = env_int("SABLE_CUT", -1);
    // all on chip only while the SMs can hold a good part of the batch at once; a batch of many waves runs faster from
    // the group-interleaved HBM workspace with many small CTAs (cfg 3: 3.5 ms vs 4.4 ms, profiles/r01_v2_sweeps.md)
    bool on_chip = gsh >= 0 && cut_env < 0;
    if (on_chip && g_env <= 0 && env_int("SABLE_THREADS", 0) <= 0) {
        const int64_t slots_sm = (int64_t)std::max<int64_t>(1, smem_sm / (need(gsh, 0, 0, 0) + 1024)) << gsh;
        if (slots_sm * n_sm * 2 < (int64_t)mb) on_chip = false;
    }
    if (on_chip) {
        ctx->placement = 0; ctx->gsh = gsh; ctx->dg_cut = ctx->pr_cut = ctx->st_cut = 0; ctx->cut_level = 0;
    } else {
        // HBM placement.  Measured (profiles/r01_v2_sweeps.md): once the batch needs many waves, resident warps and a
        // large L1 (which then holds the shared index program and Y_bus) buy more than shared-memory residency of the
        // factors, and even a small on-chip top of the elimination tree is neutral to slightly negative: everything
        // lives in the group-interleaved HBM workspace (placement 2, kernels without placement branches), the level
        // blobs are read in place (no ring), and the register file sets the CTA count (72 registers for up to 128
        // threads per CTA, 64 beyond).  SABLE_CUT=<level> asks for the mixed placement 1 (levels >= cut on chip).
        if (ctx->opt.threads <= 0 && env_int("SABLE_THREADS", 0) <= 0) th = nn <= 1200 ? 128 : nn <= 4000 ? 256 : 512;
        want_ctas = env_int("SABLE_CTAS", std::max(1, 1024 / th));
        set_ring(r_env >= 0 ? ropts[0] : RingOpt{0, 0});
        // slots per CTA (= scenarios whose HBM slices are interleaved): 4 for small grids, else 1 (measured), or SABLE_G
        int sg = 0;
        const int g_want = g_env > 0 ? g_env : (nn <= 1200 ? 4 : 1);
        while ((2 << sg) <= g_want && (g_env > 0 || ((int64_t)n_sm << (sg + 1)) <= (int64_t)std::max(mb, 1))) ++sg;
        const int cl = cut_env >= 0 ? std::min(cut_env, nl) : nl;
        const int nc = cl < nl ? T.level_ptr[cl] : nn;
        ctx->placement = cl < nl ? 1 : 2; ctx->gsh = sg; ctx->cut_level = cl;
        ctx->dg_cut = nc; ctx->pr_cut = T.pair_ptr[nc]; ctx->st_cut = cl < nl ? nc : nn + 1;
        if (ctx->placement == 1 && th <= 128) th = 256;      // the mixed kernel is built in the large variant only
        if (need(sg, ctx->dg_cut, ctx->pr_cut, ctx->st_cut) > max_optin) return fail(ctx, SABLE_ERR_INVALID_ARG, "placement does not fit shared memory");
    }
    ctx->threads = th;
    ctx->smem = (int)need(ctx->gsh, ctx->dg_cut, ctx->pr_cut, ctx->st_cut);
    ctx->front_k = 0; ctx->front_level = nl; ctx->front_f0 = nn;
    if (ctx->placement == 2) {
        // dense top front: shared memory that still leaves most of the L1 to the resident CTAs (measured budgets)
        const int kcap = env_int("SABLE_FRONT", 64);
        const int64_t budget = env_int("SABLE_FRONT_KB", th <= 128 ? 8 : th <= 256 ? 6 : 16) * 1024LL;
        if (kcap >= 2) build_front(ctx, th, ctx->gsh, budget, std::min(kcap, 96));
        if (ctx->front_k > 0) {
            ctx->front_off = align16(ctx->smem);
            ctx->smem = (int)(ctx->front_off + (mixed ? front_bytes<float>(ctx->front_k, ctx->gsh) : front_bytes<double>(ctx->front_k, ctx->gsh)));
        }
    }
    const void* fn = fused_fn(mixed, ctx->placement, th <= 128);
    CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->smem));
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, th, (size_t)ctx->smem));
    if (occ < 1) return fail(ctx, SABLE_ERR_CUDA, "NR kernel does not fit on an SM");
    occ = std::min(occ, env_int("SABLE_CTAS", occ));
    ctx->ctas_per_sm = occ; ctx->grid = occ * n_sm;
    ctx->threads1 = env_int("SABLE_THREADS1", nn <= 64 ? 32 : nn <= 1200 ? 64 : nn <= 4000 ? 256 : 512);
    return SABLE_OK;
}

extern "C" sable_status sable_create(int32_t n_bus, const int32_t* row_ptr, const int32_t* col_idx, const double* y_re,
                                     const double* y_im, const uint8_t* bus_type, int32_t slack,
                                     const sable_options* opt, sable_ctx** out) {
    sable_ctx* ctx = nullptr;      // CU() reports into g_create_err while ctx is null
    if (!out) return fail(nullptr, SABLE_ERR_INVALID_ARG, "out is NULL");
    *out = nullptr;
    sable_options o{1, SABLE_FP64, 1, SABLE_MODE_FUSED, 0, 0};
    if (opt) o = *opt;
    if (o.max_batch < 1 || (o.precision != SABLE_FP64 && o.precision != SABLE_MIXED) ||
        (o.mode != SABLE_MODE_FUSED && o.mode != SABLE_MODE_STAGED) || o.device < -1 || o.threads < 0)
        return fail(nullptr, SABLE_ERR_INVALID_ARG, "bad option value");
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
    cudaError_t e = cudaSetDevice(o.device);
    if (e != cudaSuccess) { c->err = std::string("cudaSetDevice: ") + cudaGetErrorString(e); return bail(SABLE_ERR_CUDA); }
    // packed device arrays
    std::vector<int32_t> node_bus(T.node_bus); node_bus.push_back(T.slack);
    std::vector<double2> ygb(T.ycol.size()), ydg(nn);
    for (size_t k = 0; k < T.ycol.size(); ++k) ygb[k] = make_double2(T.yg[k], T.yb[k]);
    for (int m = 0; m < nn; ++m) ydg[m] = make_double2(T.yg[T.ydiag[m]], T.yb[T.ydiag[m]]);
    std::vector<double4> py(np);
    std::vector<int2> pmj(np);
    for (int p = 0; p < np; ++p) {
        const int su = T.pair_yu[p], sl = T.pair_yl[p];
        py[p] = make_double4(su >= 0 ? T.yg[su] : 0.0, su >= 0 ? T.yb[su] : 0.0, sl >= 0 ? T.yg[sl] : 0.0, sl >= 0 ? T.yb[sl] : 0.0);
        const int m = T.pair_row[p], j = T.pair_col[p];
        pmj[p] = make_int2(m | (T.node_pq[m] ? 1 << 30 : 0), j | (T.node_pq[j] ? 1 << 30 : 0));
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
    }
    up(mm_row, &d.mm_row); up(node_bus, &d.node_bus); up(T.node_pq, &d.node_pq); up(T.yptr, &d.yptr);
    up(T.ycol, &d.ycol); up(ygb, &d.ygb); up(ydg, &d.ydiag_gb); up(pmj, &d.pair_mj); up(py, &d.pair_y);
    if (!ok) return bail(SABLE_ERR_ALLOC);
    ctx = c;
    build_blobs(T, c->lv_host, c->blob_host);
    sable_status st = choose_launch(c);
    if (st != SABLE_OK) return bail(st);
    {
        std::vector<LevelDesc> lf = build_levels(T, c->lv_host, c->threads, c->gsh, c->first_staged);
        std::vector<LevelDesc> l1 = build_levels(T, c->lv_host, c->threads1, 0, T.n_level);
        c->threads_lin = env_int("SABLE_THREADS_LIN", std::min(512, std::max(32 << c->gsh, 64)));   // 32 targets in flight per slot (measured)
        std::vector<LevelDesc> ll = build_levels(T, c->lv_host, c->threads_lin, c->gsh, T.n_level);
        up(lf, &c->level_fused); up(l1, &c->level_one); up(ll, &c->level_lin); up(c->blob_host, &d.blob);
        if (!ok) return bail(SABLE_ERR_ALLOC);
    }
    const bool mixed = o.precision == SABLE_MIXED;
    c->fac_stride = align16(mixed ? fac_bytes<float>(nn, np) : fac_bytes<double>(nn, np));
    c->work_stride = work_bytes(nn);
    auto dmalloc = [&](void** p, size_t bytes) {
        if (cudaMalloc(p, bytes) != cudaSuccess) { c->err = "device allocation failed (" + std::to_string(bytes) + " bytes)"; return false; }
        c->dev_allocs.push_back(*p); return true;
    };
    const size_t mb = (size_t)o.max_batch, nb = (size_t)T.n_bus;
    // workspace for whole groups of 1 << gsh scenarios (fused mode interleaves a group's slices; staged mode: gsh 0)
    const size_t G = (size_t)1 << c->gsh, mb_alloc = (mb + G - 1) / G * G + G;
    if (!dmalloc((void**)&c->factors, mb_alloc * c->fac_stride) || !dmalloc((void**)&c->work, mb_alloc * c->work_stride) ||
        !dmalloc((void**)&c->ints, (2 * mb + 4) * 4) || !dmalloc((void**)&c->hbuf, 9 * mb * nb * 8 + mb * 8) ||
        !dmalloc((void**)&c->hbuf_it, mb * 4) || !dmalloc((void**)&c->hbuf_cv, mb) || !dmalloc((void**)&c->zeros, nb * 8) ||
        !dmalloc((void**)&c->lbuf, 4 * mb * nb * 8))
        return bail(SABLE_ERR_ALLOC);
    if (cudaMemset(c->zeros, 0, nb * 8) != cudaSuccess || cudaMemset(c->work, 0, mb_alloc * c->work_stride) != cudaSuccess ||
        cudaMemset(c->factors, 0, mb_alloc * c->fac_stride) != cudaSuccess) { c->err = "cudaMemset failed"; return bail(SABLE_ERR_CUDA); }
    if (env_int("SABLE_TIMING", 0)) {
        const size_t tb = (4 * (size_t)T.n_level + 4) * 8;
        if (!dmalloc((void**)&c->tim, tb)) return bail(SABLE_ERR_ALLOC);
        cudaMemset(c->tim, 0, tb);
    }
    fill_info(c);
    *out = c;
    return SABLE_OK;
}

extern "C" void sable_destroy(sable_ctx* c) {
    if (!c) return;
    for (void* p : c->dev_allocs) cudaFree(p);
    delete c;
}
extern "C" const char* sable_last_error(const sable_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }
extern "C" int64_t sable_launch_count(const sable_ctx* c) { return c ? c->launches : 0; }
extern "C" sable_status sable_get_info(const sable_ctx* c, sable_info* info) {
    if (!c || !info) return SABLE_ERR_INVALID_ARG;
    *info = c->info; return SABLE_OK;
}

// ---- solve -------------------------------------------------------------------------------------------------------
template <typename T>
static cudaError_t launch_solve(sable_ctx* c, SolveArgs& A, cudaStream_t s) {
    if (c->opt.mode == SABLE_MODE_FUSED) {
        cudaError_t e = cudaMemsetAsync(A.queue, 0, 4, s);
        if (e != cudaSuccess) return e;
        A.t.level = c->level_fused;
        A.gsh = c->gsh; A.dg_cut = c->dg_cut; A.pr_cut = c->pr_cut; A.st_cut = c->st_cut;
        A.ring_r = c->ring_r; A.ring_slot = c->ring_slot; A.first_staged = c->first_staged;
        A.trash_grp = (c->opt.max_batch + (1 << c->gsh) - 1) >> c->gsh;
        A.front_k = c->front_k; A.front_f0 = c->front_f0; A.front_level = c->front_level; A.front_off = c->front_off; A.front = c->front;
        const int G = 1 << c->gsh;
        const int grid = std::min((A.batch + G - 1) / G, c->grid);
        c->factor_gsh = c->gsh;
        // the attribute is per-function state shared by every live context: set it for THIS context right before the launch
        e = cudaFuncSetAttribute(fused_fn(sizeof(T) == 4, c->placement, c->threads <= 128), cudaFuncAttributeMaxDynamicSharedMemorySize, c->smem);
        if (e != cudaSuccess) return e;
        if (c->placement == 0) k_nr_fused<T, 0, false><<<grid, c->threads, c->smem, s>>>(A);
        else if (c->placement == 1) k_nr_fused<T, 1, false><<<grid, c->threads, c->smem, s>>>(A);
        else if (c->threads <= 128) k_nr_fused<T, 2, true><<<grid, c->threads, c->smem, s>>>(A);
        else k_nr_fused<T, 2, false><<<grid, c->threads, c->smem, s>>>(A);
        c->launches += 1;
    } else {
        A.t.level = c->level_one;
        A.gsh = 0; c->factor_gsh = 0;
        k_st_init<T><<<A.batch, c->threads1, 0, s>>>(A);
        for (int i = 0; i <= A.max_it; ++i) {
            k_st_mismatch_fill<T><<<A.batch, c->threads1, 0, s>>>(A);
            if (i < A.max_it) k_st_factor_solve<T><<<A.batch, c->threads1, 0, s>>>(A);
        }
        c->launches += 2 + 2 * (int64_t)A.max_it;
    }
    return cudaGetLastError();
}

extern "C" sable_status sable_solve(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                    const double* v_set, const double* vm0, const double* va0, double tol, int32_t max_it,
                                    double* vm, double* va, int32_t* iterations, uint8_t* converged, double* final_norm,
                                    void* cuda_stream) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 0 || batch > ctx->opt.max_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch out of range");
    if (max_it < 0 || !(tol >= 0.0)) return fail(ctx, SABLE_ERR_INVALID_ARG, "max_it < 0 or tol < 0");
    ctx->have_factors = false; ctx->last_batch = batch;
    if (batch == 0) return SABLE_OK;                       /* empty batch: nothing is read or written */
    if (!p_spec || !q_spec || !v_set || !vm || !va || !iterations || !converged || ((vm0 == nullptr) != (va0 == nullptr)))
        return fail(ctx, SABLE_ERR_INVALID_ARG, "null array (vm0 and va0 must both be given or both be NULL)");
    ON_DEVICE(ctx);
    SolveArgs A{};
    A.t = ctx->d; A.batch = batch; A.max_it = max_it; A.keep = ctx->opt.keep_factors; A.tol = tol;
    A.p_spec = p_spec; A.q_spec = q_spec; A.v_set = v_set; A.vm0 = vm0; A.va0 = va0;
    A.vm = vm; A.va = va; A.final_norm = final_norm; A.iterations = iterations; A.converged = converged;
    A.factors = ctx->factors; A.work = ctx->work; A.fac_stride = ctx->fac_stride; A.work_stride = ctx->work_stride;
    A.tim = ctx->tim;
    A.queue = ctx->ints; A.status = ctx->ints + 4; A.it = ctx->ints + 4 + ctx->opt.max_batch;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    CU(ctx->opt.precision == SABLE_MIXED ? launch_solve<float>(ctx, A, s) : launch_solve<double>(ctx, A, s));
    ctx->have_factors = ctx->opt.keep_factors != 0;
    return SABLE_OK;
}

// ---- adjoint / linear solves on kept factors ---------------------------------------------------------------------
static sable_status launch_lin(sable_ctx* ctx, int batch, const double* rp, const double* rq, int transposed, double* xp,
                               double* xq, cudaStream_t s) {
    LinArgs L{};
    const int gsh = ctx->factor_gsh, G = 1 << gsh;
    L.t = ctx->d;
    L.t.level = gsh == 0 ? ctx->level_one : ctx->level_lin;
    L.batch = batch; L.transposed = transposed; L.gsh = gsh; L.rhs_p = rp; L.rhs_q = rq; L.x_p = xp; L.x_q = xq;
    L.factors = ctx->factors; L.fac_stride = ctx->fac_stride; L.work = ctx->work; L.work_stride = ctx->work_stride;
    const size_t sm = ((size_t)ctx->T.n_node * 16) << gsh;
    int max_optin = 0; CU(cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->opt.device));
    L.rhs_in_smem = sm <= std::min<size_t>((size_t)max_optin, 64 * 1024);
    const void* lin = ctx->opt.precision == SABLE_MIXED ? (const void*)k_linsolve<float> : (const void*)k_linsolve<double>;
    if (L.rhs_in_smem && sm > 48 * 1024) CU(cudaFuncSetAttribute(lin, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int th = gsh == 0 ? ctx->threads1 : ctx->threads_lin, grid = (batch + G - 1) / G;
    if (ctx->opt.precision == SABLE_MIXED) k_linsolve<float><<<grid, th, L.rhs_in_smem ? sm : 0, s>>>(L);
    else k_linsolve<double><<<grid, th, L.rhs_in_smem ? sm : 0, s>>>(L);
    ctx->launches += 1;
    CU(cudaGetLastError());
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
    return launch_lin(ctx, batch, g_va, g_vm, 1, lam_p, lam_q, (cudaStream_t)cuda_stream);
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
    const size_t sm = (size_t)ctx->T.n_bus * 16;
    R.v_in_smem = sm <= 160 * 1024;            // else the scenario's workspace slice (>= 3 (n_bus) 16 bytes) holds V
    if (R.v_in_smem && sm > 48 * 1024) CU(cudaFuncSetAttribute((const void*)k_recover, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int th = bus_threads(ctx->T.n_bus);
    k_recover<<<batch, th, R.v_in_smem ? sm : 0, (cudaStream_t)cuda_stream>>>(R);
    ctx->launches += 1;
    CU(cudaGetLastError());
    return SABLE_OK;
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
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)ctx->opt.max_batch * ctx->T.n_bus;
    LayerArgs L{};
    L.n_bus = ctx->T.n_bus; L.batch = batch; L.fptr = ctx->fptr; L.fcol = ctx->fcol; L.ftpos = ctx->ftpos; L.fgb = ctx->fgb;
    L.bus_type = ctx->d_bus_type; L.vm = vm; L.va = va; L.gl_pg = gl_pg; L.gl_qg = gl_qg; L.gl_vm = gl_vm; L.gl_va = gl_va;
    L.g_va = ctx->lbuf; L.g_vm = ctx->lbuf + n; L.lam_p = ctx->lbuf + 2 * n; L.lam_q = ctx->lbuf + 3 * n;
    L.dx_pg = dx_pg; L.dx_vm = dx_vm; L.work = ctx->work; L.work_stride = ctx->work_stride;
    const size_t sm = (size_t)ctx->T.n_bus * 48;       // V, (P, Q), row weights
    L.in_smem = sm <= 160 * 1024;          // else the scenario's workspace slice (48 n_bus bytes) holds them
    if (L.in_smem && sm > 48 * 1024) CU(cudaFuncSetAttribute((const void*)k_layer, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int th = bus_threads(ctx->T.n_bus);
    L.post = 0;
    k_layer<<<batch, th, L.in_smem ? sm : 0, s>>>(L);
    CU(cudaGetLastError());
    sable_status st = launch_lin(ctx, batch, L.g_va, L.g_vm, 1, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, s);
    if (st != SABLE_OK) return st;
    L.post = 1;
    k_layer<<<batch, th, L.in_smem ? sm : 0, s>>>(L);
    ctx->launches += 2;
    CU(cudaGetLastError());
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
    sable_status st = launch_lin(ctx, batch, g_va, g_vm, 1, lam_p, lam_q, s);
    if (st != SABLE_OK || sweeps == 0) return st;
    const size_t n = (size_t)ctx->opt.max_batch * ctx->T.n_bus, nb = (size_t)batch * ctx->T.n_bus;
    LayerArgs L{};
    L.n_bus = ctx->T.n_bus; L.batch = batch; L.fptr = ctx->fptr; L.fcol = ctx->fcol; L.ftpos = ctx->ftpos; L.fgb = ctx->fgb;
    L.bus_type = ctx->d_bus_type; L.vm = vm; L.va = va; L.gl_va = g_va; L.gl_vm = g_vm; L.lam_p = lam_p; L.lam_q = lam_q;
    L.g_va = ctx->lbuf; L.g_vm = ctx->lbuf + n; L.work = ctx->work; L.work_stride = ctx->work_stride; L.post = 2;
    const size_t sm = (size_t)ctx->T.n_bus * 48;       // V, (P, Q), row weights
    L.in_smem = sm <= 160 * 1024;
    if (L.in_smem && sm > 48 * 1024) CU(cudaFuncSetAttribute((const void*)k_layer, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
    const int th = bus_threads(ctx->T.n_bus);
    for (int it = 0; it < sweeps; ++it) {
        k_layer<<<batch, th, L.in_smem ? sm : 0, s>>>(L);                                   // r = g - J1^T lambda   (FP64)
        CU(cudaGetLastError());
        st = launch_lin(ctx, batch, L.g_va, L.g_vm, 1, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, s);   // J1^T d = r  (kept factors)
        if (st != SABLE_OK) return st;
        k_add2<<<(int)std::min<size_t>((nb + 255) / 256, 4096), 256, 0, s>>>(lam_p, lam_q, ctx->lbuf + 2 * n, ctx->lbuf + 3 * n, nb);
        CU(cudaGetLastError());
        ctx->launches += 2;
    }
    return SABLE_OK;
}

// ---- host-buffer wrappers (end-to-end path: H2D, solve, D2H; synchronous) ------------------------------------------
extern "C" sable_status sable_solve_host(sable_ctx* ctx, int32_t batch, const double* p_spec, const double* q_spec,
                                         const double* v_set, const double* vm0, const double* va0, double tol,
                                         int32_t max_it, double* vm, double* va, int32_t* iterations, uint8_t* converged,
                                         double* final_norm) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 0 || batch > ctx->opt.max_batch) return fail(ctx, SABLE_ERR_INVALID_ARG, "batch out of range");
    if (!p_spec || !q_spec || !v_set || !vm || !va || !iterations || !converged || ((vm0 == nullptr) != (va0 == nullptr)))
        return fail(ctx, SABLE_ERR_INVALID_ARG, "null array");
    if (batch == 0) { ctx->have_factors = false; ctx->last_batch = 0; return SABLE_OK; }
    ON_DEVICE(ctx);
    const size_t n = (size_t)batch * ctx->T.n_bus, bytes = n * 8;
    double* d = ctx->hbuf;       // slots: 0 p, 1 q, 2 vset, 3 vm0, 4 va0, 5 vm, 6 va, (7, 8 adjoint), then norm
    double* dn = ctx->hbuf + 9 * (size_t)ctx->opt.max_batch * ctx->T.n_bus;
    CU(cudaMemcpyAsync(d, p_spec, bytes, cudaMemcpyHostToDevice, 0));
    CU(cudaMemcpyAsync(d + n, q_spec, bytes, cudaMemcpyHostToDevice, 0));
    CU(cudaMemcpyAsync(d + 2 * n, v_set, bytes, cudaMemcpyHostToDevice, 0));
    if (vm0) { CU(cudaMemcpyAsync(d + 3 * n, vm0, bytes, cudaMemcpyHostToDevice, 0)); CU(cudaMemcpyAsync(d + 4 * n, va0, bytes, cudaMemcpyHostToDevice, 0)); }
    sable_status st = sable_solve(ctx, batch, d, d + n, d + 2 * n, vm0 ? d + 3 * n : nullptr, vm0 ? d + 4 * n : nullptr, tol, max_it,
                                  d + 5 * n, d + 6 * n, ctx->hbuf_it, ctx->hbuf_cv, dn, nullptr);
    if (st != SABLE_OK) return st;
    CU(cudaMemcpyAsync(vm, d + 5 * n, bytes, cudaMemcpyDeviceToHost, 0));
    CU(cudaMemcpyAsync(va, d + 6 * n, bytes, cudaMemcpyDeviceToHost, 0));
    CU(cudaMemcpyAsync(iterations, ctx->hbuf_it, (size_t)batch * 4, cudaMemcpyDeviceToHost, 0));
    CU(cudaMemcpyAsync(converged, ctx->hbuf_cv, (size_t)batch, cudaMemcpyDeviceToHost, 0));
    if (final_norm) CU(cudaMemcpyAsync(final_norm, dn, (size_t)batch * 8, cudaMemcpyDeviceToHost, 0));
    CU(cudaStreamSynchronize(0));
    return SABLE_OK;
}

extern "C" sable_status sable_adjoint_host(sable_ctx* ctx, int32_t batch, const double* g_va, const double* g_vm,
                                           double* lam_p, double* lam_q) {
    if (!ctx) return SABLE_ERR_INVALID_ARG;
    if (ctx->opt.device < 0) return fail(ctx, SABLE_ERR_STATE, "host-only context");
    if (batch < 0 || batch > ctx->opt.max_batch || !g_va || !g_vm || !lam_p || !lam_q) return fail(ctx, SABLE_ERR_INVALID_ARG, "bad argument");
    if (batch == 0) return SABLE_OK;
    ON_DEVICE(ctx);
    const size_t n = (size_t)batch * ctx->T.n_bus, bytes = n * 8;
    double* d = ctx->hbuf;
    CU(cudaMemcpyAsync(d, g_va, bytes, cudaMemcpyHostToDevice, 0));
    CU(cudaMemcpyAsync(d + n, g_vm, bytes, cudaMemcpyHostToDevice, 0));
    sable_status st = sable_adjoint(ctx, batch, d, d + n, d + 7 * n, d + 8 * n, nullptr);
    if (st != SABLE_OK) return st;
    CU(cudaMemcpyAsync(lam_p, d + 7 * n, bytes, cudaMemcpyDeviceToHost, 0));
    CU(cudaMemcpyAsync(lam_q, d + 8 * n, bytes, cudaMemcpyDeviceToHost, 0));
    CU(cudaStreamSynchronize(0));
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
    D.t = ctx->d; D.t.level = ctx->level_one; D.zeros = ctx->zeros; ctx->factor_gsh = 0;
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
    ctx->have_factors = false;
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
    return launch_lin(ctx, batch, rhs_p, rhs_q, transpose ? 1 : 0, x_p, x_q, (cudaStream_t)cuda_stream);
}
