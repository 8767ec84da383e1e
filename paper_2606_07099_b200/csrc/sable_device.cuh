// Device-side view of the shared fixed-pattern template and of one scenario slot's storage.
//
// Block conventions.  Every non-slack bus is a node with a 2x2 block: rows (P_m, Q_m), columns (theta_m, Vm_m),
// stored row-major [dP/dth, dP/dVm, dQ/dth, dQ/dVm].  A PV node keeps the block with the Q row and Vm column padded
// (0 off the diagonal, 1 on it).  Per scenario the factor storage is, in units of one block (4 values of T):
//   dg[n_node]     : J(m,m), then after refactor the INVERSE of the pivot block D_m
//   pr[2*n_pair]   : pair p = (m,j), m < j:  pr[2p] = J(m,j) -> U(m,j);  pr[2p+1] = J(j,m) -> L(j,m)
// and the state, three 16-byte records per node (index n_node = slack):
//   vv = (V_re, V_im)   ma = (|V|, theta)   rh = (rhs_P/theta, rhs_Q/Vm): -F, then y, then dz (g, w, lambda: adjoint)
//
// Placement.  A CTA works on G = 2^gsh scenarios in lockstep ("slots"; thread tid serves slot g = tid % G).  The late
// part of every array (nodes >= cut, pairs >= cut: the top of the elimination tree, where levels are narrow and
// latency decides) lives in shared memory, interleaved over the slots in 16-byte vectors:
//   address = base + ((index_in_vectors << gsh) + g) * 16
// so that the G lanes serving one target read consecutive 16-byte words (conflict-free LDS.128).  The early part lives
// in the HBM workspace of the scenario's GROUP (scenarios b with equal b >> gsh), interleaved over the group in the same
// way -- a warp then touches 16 G contiguous bytes per target instead of 32 scattered sectors (coalesced LDG.128; the
// L1 wavefront count, which bounded the scenario-major layout at 65 % of its peak, drops by up to G) -- and that is also
// where kept factors are handed to sable_adjoint.  With gsh = 0 (staged / debug kernels) this is a plain contiguous
// slice per scenario.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sable {

// One elimination level: node range [m0, m1), the pairs those nodes own [p0, p1), the lane split per target, and the
// level's slice of the index program ("blob": everything the factor / forward / backward phases of this level read
// besides values).  Blob layout (byte offsets from the blob start; counts nm = m1 - m0, np = p1 - p0):
//   int32 dptr[nm+1]   diag target i subtracts the terms dak[dptr[i] .. dptr[i+1])
//   int32 tptr[np+1]   pair target i subtracts the terms tab[tptr[i] .. tptr[i+1])
//   int32 pptr[nm+1]   node i owns the pairs p0 + [pptr[i] & kIdxMask, pptr[i+1] & kIdxMask); bit 30 of pptr[i] = PQ node
//   int2  dak[]        (pair (k,m), node k)                                  at o_dak
//   int2  pmj[np]      (m | pq_m << 30, j | pq_j << 30)                      at o_pmj
//   int2  tab[]        (pair (k,m), pair (k,j))                              at o_tab
// Narrow levels (staged = 1) are streamed through a shared-memory ring by cp.async.bulk one or two levels ahead of
// use, so that no index load of the latency-critical top of the elimination tree goes to L2; wide levels are read
// in place (their latency hides behind the many targets in flight).
struct LevelDesc {
    int32_t m0, m1, p0, p1;
    uint8_t sd, sp, sb, staged;   // diag / pair / backward lane splits (lanes per target = 1 << s)
    int32_t blob_off, blob_bytes; // slice of DevTemplate::blob (16-byte aligned, size a multiple of 16)
    int32_t o_tptr, o_pptr, o_dak, o_pmj, o_tab, o_py;   // o_py: end of the lists (the front's descriptor keeps one more list there)
    int32_t pad;
};

struct RowClass { int32_t i0, i1, ssh; };   // rows mm_order[i0 .. i1) of the mismatch pass are served by 1 << ssh lanes each

struct DevTemplate {
    int32_t n_bus, n_node, n_pair, n_level, slack;
    int32_t n_class;            // mismatch pass: nodes sorted by Y-row length, long rows split over lanes
    RowClass mm_class[6];
    const int4* mm_row;         // [n_node] (node m, first Y slot, end Y slot, bus | pq << 30), longest rows first
    const LevelDesc* level;     // [n_level]
    const char* blob;           // level slices of the index program
    const int32_t* node_bus;    // [n_node+1]  (entry n_node = slack bus)
    const uint8_t* node_pq;     // [n_node]
    const int32_t* yptr;        // [n_node+1]  Y rows of the non-slack buses in node order
    const int32_t* ycol;        // node positions (slack = n_node)
    const double2* ygb;         // (G, B) per stored Y entry
    const double2* ydiag_gb;    // [n_node] (G_mm, B_mm)
    const int2*    pair_mj;     // [n_pair] (m | pq_m << 30, j | pq_j << 30)   (separate fill pass only)
    const double4* pair_y;      // [n_pair]                                     (separate fill pass only)
};
constexpr int kIdxMask = 0x3fffffff;

template <typename T> struct Blk { T a, b, c, d; };   // [[a b][c d]]

// acc -= x * y  (2x2)
template <typename T> __device__ __forceinline__ void mulsub(Blk<T>& acc, const Blk<T>& x, const Blk<T>& y) {
    acc.a -= x.a * y.a + x.b * y.c;  acc.b -= x.a * y.b + x.b * y.d;
    acc.c -= x.c * y.a + x.d * y.c;  acc.d -= x.c * y.b + x.d * y.d;
}
template <typename T> __device__ __forceinline__ Blk<T> mul(const Blk<T>& x, const Blk<T>& y) {
    return {x.a * y.a + x.b * y.c, x.a * y.b + x.b * y.d, x.c * y.a + x.d * y.c, x.c * y.b + x.d * y.d};
}
template <typename T> __device__ __forceinline__ Blk<T> inv(const Blk<T>& x) {
    T det = x.a * x.d - x.b * x.c, r = T(1) / det;
    return {x.d * r, -x.b * r, -x.c * r, x.a * r};
}
template <typename T> __device__ __forceinline__ T shx(T v, int o) { return __shfl_xor_sync(0xffffffffu, v, o); }
template <typename T> __device__ __forceinline__ void blk_add_shx(Blk<T>& v, int o) {
    v.a += shx(v.a, o); v.b += shx(v.b, o); v.c += shx(v.c, o); v.d += shx(v.d, o);
}

// 16-byte vector access to one block of T at p; the second vector of an FP64 block is `vs` bytes further
__device__ __forceinline__ Blk<double> ld_blk(const double* p, int vs) {
    const double2 x = *reinterpret_cast<const double2*>(p);
    const double2 y = *reinterpret_cast<const double2*>(reinterpret_cast<const char*>(p) + vs);
    return {x.x, x.y, y.x, y.y};
}
__device__ __forceinline__ Blk<float> ld_blk(const float* p, int) {
    const float4 x = *reinterpret_cast<const float4*>(p);
    return {x.x, x.y, x.z, x.w};
}
__device__ __forceinline__ void st_blk(double* p, int vs, const Blk<double>& v) {
    *reinterpret_cast<double2*>(p) = make_double2(v.a, v.b);
    *reinterpret_cast<double2*>(reinterpret_cast<char*>(p) + vs) = make_double2(v.c, v.d);
}
__device__ __forceinline__ void st_blk(float* p, int, const Blk<float>& v) {
    *reinterpret_cast<float4*>(p) = make_float4(v.a, v.b, v.c, v.d);
}

// One thread's view of the slot it serves.  kP = 0: everything in shared memory; 2: everything in the HBM workspace
// (both without placement branches); 1: mixed, split at the cuts.
template <typename T, int kP> struct Slot {
    static constexpr int VPB = (int)(4 * sizeof(T) / 16);      // 16-byte vectors per block: 2 (FP64) or 1 (FP32)
    // Three per-thread pointers (shared base, factor slice and state slice of the group, each offset by g * 16) plus
    // CTA-uniform byte offsets of the arrays behind them (uniform registers / constant bank: keeps the register count
    // of the persistent kernel down).  Shared order: vv | ma | rh | dg | pr.  HBM: factors = dg | pr, state = vv | ma | rh.
    char *sb, *gf, *gw;
    unsigned so_ma, so_rh, so_dg, so_pr, go_pr, go_ma, go_rh;
    int dg_cut, pr_cut, st_cut, gsh;                          // node cut of dg, pair cut of pr, node cut of vv/ma/rh
    __device__ __forceinline__ char* s_vv() const { return sb; }
    __device__ __forceinline__ char* s_ma() const { return sb + so_ma; }
    __device__ __forceinline__ char* s_rh() const { return sb + so_rh; }
    __device__ __forceinline__ char* s_dg() const { return sb + so_dg; }
    __device__ __forceinline__ char* s_pr() const { return sb + so_pr; }
    __device__ __forceinline__ char* g_dg() const { return gf; }
    __device__ __forceinline__ char* g_pr() const { return gf + go_pr; }
    __device__ __forceinline__ char* g_vv() const { return gw; }
    __device__ __forceinline__ char* g_ma() const { return gw + go_ma; }
    __device__ __forceinline__ char* g_rh() const { return gw + go_rh; }

    // byte offsets are 32-bit: a group's slice (and shared memory) is far below 4 GB
    __device__ __forceinline__ T* blk_ptr(char* sb, char* gb, int idx, int cut_blocks, int& vs) const {
        vs = 16 << gsh;
        if (kP == 0) return reinterpret_cast<T*>(sb + ((unsigned)(idx * VPB) << (gsh + 4)));
        if (kP == 1 && idx >= cut_blocks) return reinterpret_cast<T*>(sb + ((unsigned)((idx - cut_blocks) * VPB) << (gsh + 4)));
        return reinterpret_cast<T*>(gb + ((unsigned)(idx * VPB) << (gsh + 4)));
    }
    __device__ __forceinline__ Blk<T> ldD(int m) const { int vs; const T* p = blk_ptr(s_dg(), g_dg(), m, dg_cut, vs); return ld_blk(p, vs); }
    __device__ __forceinline__ void stD(int m, const Blk<T>& v) const { int vs; T* p = blk_ptr(s_dg(), g_dg(), m, dg_cut, vs); st_blk(p, vs, v); }
    __device__ __forceinline__ Blk<T> ldU(int p) const { int vs; const T* q = blk_ptr(s_pr(), g_pr(), 2 * p, 2 * pr_cut, vs); return ld_blk(q, vs); }
    __device__ __forceinline__ Blk<T> ldL(int p) const { int vs; const T* q = blk_ptr(s_pr(), g_pr(), 2 * p + 1, 2 * pr_cut, vs); return ld_blk(q, vs); }
    __device__ __forceinline__ void stU(int p, const Blk<T>& v) const { int vs; T* q = blk_ptr(s_pr(), g_pr(), 2 * p, 2 * pr_cut, vs); st_blk(q, vs, v); }
    __device__ __forceinline__ void stL(int p, const Blk<T>& v) const { int vs; T* q = blk_ptr(s_pr(), g_pr(), 2 * p + 1, 2 * pr_cut, vs); st_blk(q, vs, v); }

    __device__ __forceinline__ double2* st_ptr(char* sb, char* gb, int m) const {
        if (kP == 0) return reinterpret_cast<double2*>(sb + ((unsigned)m << (gsh + 4)));
        if (kP == 1 && m >= st_cut) return reinterpret_cast<double2*>(sb + ((unsigned)(m - st_cut) << (gsh + 4)));
        return reinterpret_cast<double2*>(gb + ((unsigned)m << (gsh + 4)));
    }
    __device__ __forceinline__ double2 vv(int m) const { return *st_ptr(s_vv(), g_vv(), m); }
    __device__ __forceinline__ double2 ma(int m) const { return *st_ptr(s_ma(), g_ma(), m); }
    __device__ __forceinline__ double2 rh(int m) const { return *st_ptr(s_rh(), g_rh(), m); }
    __device__ __forceinline__ void set_vv(int m, double2 v) const { *st_ptr(s_vv(), g_vv(), m) = v; }
    __device__ __forceinline__ void set_ma(int m, double2 v) const { *st_ptr(s_ma(), g_ma(), m) = v; }
    __device__ __forceinline__ void set_rh(int m, double2 v) const { *st_ptr(s_rh(), g_rh(), m) = v; }
};

// ---- level-blob ring: cp.async.bulk (TMA 1-D bulk copy) + mbarrier ------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* b, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* b) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, uint32_t parity) {
    asm volatile("{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
                 ::"r"(smem_u32(b)), "r"(parity) : "memory");
}

// The staged levels [first, n_level) are visited forward then backward, once per sweep pair; entry e of that endless
// sequence lives in ring slot e % R.  Thread 0 is the producer; every thread consumes and tracks `use` itself.
struct BlobRing {
    char* slots; unsigned long long* mbar;
    const char* gblob; const LevelDesc* lv;
    int R, slot_bytes, first, n_level;
    bool on;                   // false (a compile-time constant in the HBM-placement kernels): blobs are read in place
    unsigned use;
    unsigned long long* tim;   // optional per-phase cycle counters of CTA 0 (sable_debug_timing); nullptr = off
    __device__ __forceinline__ void tick(int slot, long long& t0) const {   // thread 0 of CTA 0, right after a barrier
        if (tim && threadIdx.x == 0) { const long long t1 = clock64(); tim[slot] += (unsigned long long)(t1 - t0); t0 = t1; }
    }
    __device__ __forceinline__ int level_of(unsigned e) const {
        const int ns = n_level - first, r = (int)(e % (unsigned)(2 * ns));
        return r < ns ? first + r : n_level - 1 - (r - ns);
    }
    __device__ __forceinline__ void issue(unsigned e) const {          // producer thread only
        const LevelDesc& d = lv[level_of(e)];
        const int sl = (int)(e % (unsigned)R);
        mbar_expect_tx(mbar + sl, (uint32_t)d.blob_bytes);
        bulk_g2s(slots + (size_t)sl * slot_bytes, gblob + d.blob_off, (uint32_t)d.blob_bytes, mbar + sl);
    }
    __device__ __forceinline__ void start() {                          // all threads, once; contains a barrier
        use = 0;
        if (!on) return;
        if (first < n_level && threadIdx.x == 0) {
            for (int i = 0; i < R; ++i) mbar_init(mbar + i, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        }
        __syncthreads();
        if (first < n_level && threadIdx.x == 0) for (int i = 0; i < R; ++i) issue((unsigned)i);
    }
    __device__ __forceinline__ const char* acquire(int l, const LevelDesc& d) const {
        if (!on || l < first) return gblob + d.blob_off;
        const int sl = (int)(use % (unsigned)R);
        mbar_wait(mbar + sl, (use / (unsigned)R) & 1u);
        return slots + (size_t)sl * slot_bytes;
    }
    // after a CTA barrier that follows the last read of level l's blob
    __device__ __forceinline__ void release(int l) {
        if (!on || l < first) return;
        if (threadIdx.x == 0) issue(use + (unsigned)R);
        ++use;
    }
    // a backward sweep that is not run: its entries still pass through the ring (the producer runs R entries ahead),
    // so consume them; contains barriers
    __device__ __forceinline__ void skip_sweep() {
        if (!on) return;
        for (int l = n_level - 1; l >= first; --l) {
            const int sl = (int)(use % (unsigned)R);
            mbar_wait(mbar + sl, (use / (unsigned)R) & 1u);
            __syncthreads();
            release(l);
        }
    }
    __device__ __forceinline__ void drain() const {                    // before the CTA exits: no copy may be in flight
        if (on && first < n_level && threadIdx.x == 0)
            for (unsigned e = use; e < use + (unsigned)R; ++e) mbar_wait(mbar + (e % (unsigned)R), (e / (unsigned)R) & 1u);
    }
};

__device__ __forceinline__ double nan_max(double x, double y) {   // NaN-propagating max of non-negative values
    return (x != x || y != y) ? __longlong_as_double(0x7ff8000000000000LL) : fmax(x, y);
}

// Per-slot CTA-wide max (a NaN anywhere in slot g gives NaN for g, reading 18).  `red` holds
// (blockDim.x / 32) * 32 doubles.  Every thread returns the max over the threads that serve its slot.  Two barriers.
__device__ __forceinline__ double slot_max_nan(double v, double* red, int gsh) {
    for (int o = 16; o >= (1 << gsh); o >>= 1) v = nan_max(v, __shfl_xor_sync(0xffffffffu, v, o));
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = blockDim.x >> 5, g = threadIdx.x & ((1 << gsh) - 1);
    __syncthreads();
    if (l < (1 << gsh)) red[w * 32 + l] = v;
    __syncthreads();
    double r = red[g];
    for (int i = 1; i < nw; ++i) r = nan_max(r, red[i * 32 + g]);
    return r;
}

}  // namespace sable
