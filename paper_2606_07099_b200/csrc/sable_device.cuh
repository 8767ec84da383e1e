// Device-side view of the shared fixed-pattern template and of one scenario slot's storage.
//
// Block conventions.  Every non-slack bus is a node with a 2x2 block: rows (P_m, Q_m), columns (theta_m, Vm_m),
// stored row-major [dP/dth, dP/dVm, dQ/dth, dQ/dVm].  A PV node keeps the block with the Q row and Vm column padded
// (0 off the diagonal, 1 on it).  The factorisation is kept in the form  J1 = L' D^-1 U  (L' = the UNSCALED lower
// blocks, U upper blocks, D the pivot blocks):  per scenario, in units of one block (4 values of T),
//   dg[n_node]   : J(m,m), then after refactor the INVERSE of the pivot block D_m
//   pu[n_pair]   : pair p = (m,j), m < j:  J(m,j) -> U(m,j)
//   pl[n_pair]   :                         J(j,m) -> L'(j,m) = J(j,m) - sum_k L'(j,k) D_k^-1 U(k,m)
// (U and L' in two separate arrays: a triangular sweep streams whole sectors of the one it needs) and the state,
// three 16-byte records per node (index n_node = slack):
//   vv = (V_re, V_im)   ma = (|V|, theta)   rh = (rhs_P/theta, rhs_Q/Vm): -F, then z = D^-1 y, then dz (g, w, lambda: adjoint)
// Keeping L' unscaled removes the "scale by D_m^-1" phase (and its barrier) from every elimination level: a consumer
// multiplies by D_k^-1 of the eliminated node k on the fly (one more L1-resident block per term).
//
// Placement.  A CTA works on G = 2^gsh scenarios in lockstep ("slots"; thread tid serves slot g = tid % G).  Either
// every array of every slot lives in shared memory (kP = 0), interleaved over the slots in 16-byte vectors:
//   address = base + ((index_in_vectors << gsh) + g) * 16
// so that the G lanes serving one target read consecutive 16-byte words (conflict-free LDS.128), or (kP = 2) in the HBM
// workspace of the scenario's GROUP (scenarios b with equal b >> gsh), interleaved over the group in the same way -- a
// warp then touches 16 G contiguous bytes per target instead of 32 scattered sectors (coalesced LDG.128) -- and that is
// also where kept factors are handed to sable_adjoint.  With gsh = 0 this is a plain contiguous slice per scenario.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sable {

// Targets of one kind (diagonal targets or pair targets) of a level, sorted by descending list length, are cut into
// classes; the targets [start, i1) of a class are served by 1 << ssh lanes each (per slot).  A warp-sized group of
// targets of one class is a TASK; the tasks of a level (diagonal classes first) are dealt to the warps round-robin, so a
// narrow level costs every warp at most one dependent chain.
struct Cls { int32_t start, i1; uint8_t ssh, diag; uint16_t pad; };
constexpr int kMaxCls = 3;      // per kind
// 1: a pair target is served as two block-targets (U half, L' half: three operand blocks per item and lane);
// 0: as one target with both accumulators (five operand blocks per item and lane)
#ifndef SABLE_HALF_TARGETS
#define SABLE_HALF_TARGETS 0
#endif
constexpr int kTargetUnit = SABLE_HALF_TARGETS ? 2 : 1;

// One elimination level: node range [m0, m1), the pairs those nodes own [p0, p1), and the level's slice of the index
// program ("blob": everything the factor / forward / backward phases of this level read besides values).  Blob layout
// (byte offsets from the blob start; counts nm = m1 - m0, np = p1 - p0):
//   int32 dptr[nm+1]   the diag target at SORTED position i (descending list length) subtracts dak[dptr[i] .. dptr[i+1])
//   int32 dord[nm]     local node index (m - m0) of sorted position i                       at o_dord
//   int32 tptr[np+1]   the pair target at SORTED position i (descending list length) subtracts tab[tptr[i] .. tptr[i+1])
//   int32 tord[np]     local pair index (p - p0) of sorted position i, | kFromZero for a fill-in   at o_tord
//                      pair (no Y entry: J(m,j) = J(j,m) = 0, nothing is stored for it before the refactor)
//   int32 pptr[nm+1]   node i owns the pairs p0 + [pptr[i], pptr[i+1])                        at o_pptr
//   int2  dak[]        (pair a = (k,m), node k)                                             at o_dak
//   int2  pmj[np]      (m | pq_m << 30, j | pq_j << 30)                                     at o_pmj
//   int4  tab[]        (pair a = (k,m), pair b = (k,j), node k, 0)                          at o_tab
// Pair target (m,j):  U(m,j) -= L'(a) D_k^-1 U(b);  L'(j,m) -= L'(b) D_k^-1 U(a)   per item.
struct LevelDesc {
    int32_t m0, m1, p0, p1;
    int32_t blob_off, blob_bytes;     // slice of DevTemplate::blob (16-byte aligned, size a multiple of 16)
    int32_t o_dord, o_tptr, o_tord, o_pptr, o_dak, o_pmj, o_tab;
    uint8_t sb, n_cls, staged, pad;   // backward lane split; classes in use (diagonal classes first); staged: streamed through the blob ring
    int32_t n_big;                    // the first n_big diag targets are "big": served by every warp of the CTA in turn
    Cls cls[2 * kMaxCls];
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
    const int32_t* ycol;        // per stored Y entry: column node position (slack = n_node)
    const int2*    ycd;         // the same with the walk's destination: (column node position (slack = n_node), destination of the Jacobian
                                // block J(row, column): pair p | half << 29 (0: U, 1: L') | column is PQ << 30; -1: none)
    const double2* ygb;         // (G, B) per stored Y entry
    int32_t n_jpair;            // pairs with a Y entry (the others are fill-in), for the pair-pass form of a2:
    const int4*    jp_mj;       // [n_jpair] (m | pq_m << 30, j | pq_j << 30, pair p, 0)
    const double4* jp_y;        // [n_jpair] (G_mj, B_mj, G_jm, B_jm)
    const double2* ydiag_gb;    // [n_node] (G_mm, B_mm)
};
constexpr int kIdxMask = 0x3fffffff;
constexpr int kPairMask = 0x1fffffff;   // pair index of a ycd destination
constexpr int kFromZero = 1 << 30;      // tord flag

template <typename T> struct Blk { T a, b, c, d; };   // [[a b][c d]]

// acc -= x * y  (2x2)
template <typename T> __device__ __forceinline__ void mulsub(Blk<T>& acc, const Blk<T>& x, const Blk<T>& y) {
    acc.a -= x.a * y.a + x.b * y.c;  acc.b -= x.a * y.b + x.b * y.d;
    acc.c -= x.c * y.a + x.d * y.c;  acc.d -= x.c * y.b + x.d * y.d;
}
template <typename T> __device__ __forceinline__ Blk<T> mul(const Blk<T>& x, const Blk<T>& y) {
    return {x.a * y.a + x.b * y.c, x.a * y.b + x.b * y.d, x.c * y.a + x.d * y.c, x.c * y.b + x.d * y.d};
}
// Inverse of a pivot block.  There is no pivot search (the pattern is shared by the batch): a block whose determinant
// is tiny against its largest entry squared -- |det| <= eps * max|entry|^2, i.e. a condition number above 1 / eps, or a
// non-finite determinant -- is FLAGGED through `bad` and the caller reports it per scenario (sable.h:
// sable_get_pivot_flags).  eps = 1e-10 in FP64, 1e-6 with FP32 factors (the identity-padded block of a PV node has the
// condition number |dP/dtheta| <= ~1e4, which must not trip the flag).
template <typename T> __device__ __forceinline__ T pivot_eps();
template <> __device__ __forceinline__ double pivot_eps<double>() { return 1e-10; }
template <> __device__ __forceinline__ float pivot_eps<float>() { return 1e-6f; }
template <typename T> __device__ __forceinline__ Blk<T> inv(const Blk<T>& x, bool& bad) {
    const T det = x.a * x.d - x.b * x.c, r = T(1) / det;
    const T n = fmax(fmax(fabs(x.a), fabs(x.b)), fmax(fabs(x.c), fabs(x.d)));
    bad |= !(fabs(det) > pivot_eps<T>() * n * n);
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
// whole block in one access (HBM workspace: blocks are interleaved over the slots as units of 4 sizeof(T) bytes): one
// 256-bit load / store per FP64 block (sm_100: LDG.256 / STG.256) -- half the L1 wavefronts of two 128-bit accesses
// Cache hints of the factor blocks in the HBM workspace (SABLE_FAC_HINT = 0 switches them off): a scenario's factors are a
// stream several times its SM's share of the L2 and far beyond the L1 -- loads do not allocate in the L1 (which stays with
// the state gathers and the index program), stores are first in line for eviction from the L2.  Measured on the B200: cfg 3
// 2.07 -> 2.03 ms, cfg 5 5.00 -> 4.85, mesh 3.66 -> 3.56, adjoint on the mesh 0.445 -> 0.40; other combinations
// (L2::evict_first on the loads, L1 / L2 evict_last on the state gathers) were neutral or slower.
#ifndef SABLE_FAC_HINT
#define SABLE_FAC_HINT 1
#endif
#if SABLE_FAC_HINT
#define SABLE_FAC_LD ".L1::no_allocate"
#define SABLE_FAC_ST ".L2::evict_first"
#else
#define SABLE_FAC_LD ""
#define SABLE_FAC_ST ""
#endif
__device__ __forceinline__ Blk<double> ldg_blk(const double* p) {
    Blk<double> v;
    asm volatile("ld.global" SABLE_FAC_LD ".v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.a), "=d"(v.b), "=d"(v.c), "=d"(v.d) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ Blk<float> ldg_blk(const float* p) {
#if SABLE_FAC_HINT
    Blk<float> v;
    asm volatile("ld.global.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.a), "=f"(v.b), "=f"(v.c), "=f"(v.d) : "l"(p) : "memory");
    return v;
#else
    return ld_blk(p, 0);
#endif
}
__device__ __forceinline__ void stg_blk(double* p, const Blk<double>& v) {
    asm volatile("st.global" SABLE_FAC_ST ".v4.f64 [%0], {%1,%2,%3,%4};" ::"l"(p), "d"(v.a), "d"(v.b), "d"(v.c), "d"(v.d) : "memory");
}
__device__ __forceinline__ void stg_blk(float* p, const Blk<float>& v) { st_blk(p, 0, v); }

// One thread's view of the slot it serves.  kP = 0: everything in shared memory; 2: everything in the HBM workspace
// (two kernel families without placement branches).
template <typename T, int kP> struct Slot {
    static constexpr int VPB = (int)(4 * sizeof(T) / 16);      // 16-byte vectors per block: 2 (FP64) or 1 (FP32)
    // Per-thread base pointers (shared base; factor slice and state slice of the group; each offset by g * 16) plus
    // CTA-uniform byte offsets of the arrays behind them.  Order in both memories: factors = dg | pu | pl, state = vv | ma | rh
    // (shared: state first, then factors).
    char *sb, *gf, *gw;
    unsigned so_ma, so_rh, so_dg, so_pu, so_pl, go_pu, go_pl, go_ma, go_rh;
    int gsh;
    // byte offsets are 32-bit: a group's slice (and shared memory) is far below 4 GB.  Shared memory: blocks interleaved
    // over the slots in 16-byte vectors (sb carries g * 16); HBM: interleaved as whole blocks (gf carries g * kBlk).
    static constexpr int kBlk = (int)(4 * sizeof(T));
#ifdef SABLE_BOUNDS
    // debug build (-DSABLE_BOUNDS): every block / state access is checked against the array it addresses; a violation traps
    // (compute-sanitizer is closed on the measurement pool: profiles/r02_sanitizer.md)
    int nn_, np_;
    __device__ __forceinline__ void chk_blk(unsigned go, int idx) const {
        const int n = go == 0u ? nn_ : np_;
        if (idx < 0 || idx >= n || (go != 0u && go != go_pu && go != go_pl)) __trap();
    }
    __device__ __forceinline__ void chk_st(int m) const { if (m < 0 || m > nn_) __trap(); }
#else
    __device__ __forceinline__ void chk_blk(unsigned, int) const {}
    __device__ __forceinline__ void chk_st(int) const {}
#endif
    __device__ __forceinline__ Blk<T> ldB(unsigned so, unsigned go, int idx) const {
        chk_blk(kP == 0 ? (so == so_dg ? 0u : so == so_pu ? go_pu : go_pl) : go, idx);
        if (kP == 0) return ld_blk(reinterpret_cast<const T*>(sb + (so + ((unsigned)(idx * VPB) << (gsh + 4)))), 16 << gsh);
        return ldg_blk(reinterpret_cast<const T*>(gf + (go + (((unsigned)idx << gsh) * kBlk))));
    }
    __device__ __forceinline__ void stB(unsigned so, unsigned go, int idx, const Blk<T>& v) const {
        chk_blk(kP == 0 ? (so == so_dg ? 0u : so == so_pu ? go_pu : go_pl) : go, idx);
        if (kP == 0) st_blk(reinterpret_cast<T*>(sb + (so + ((unsigned)(idx * VPB) << (gsh + 4)))), 16 << gsh, v);
        else stg_blk(reinterpret_cast<T*>(gf + (go + (((unsigned)idx << gsh) * kBlk))), v);
    }
    __device__ __forceinline__ Blk<T> ldD(int m) const { return ldB(so_dg, 0u, m); }
    __device__ __forceinline__ void stD(int m, const Blk<T>& v) const { stB(so_dg, 0u, m, v); }
    // Pairs.  HBM workspace with FP32 factors: U and L' of a pair sit side by side in one 32-byte RECORD (one 256-bit access
    // moves both: an item of the refactor needs both blocks of each of its pairs -- 3 loads per pair item instead of 5); with
    // FP64 factors (a block is 32 bytes already) and in shared memory they are two arrays.  gpx: extra lane offset of the
    // record interleave (records are twice as wide as the blocks gf is offset for).
    static constexpr bool kPairRec = kP == 2 && sizeof(T) == 4;
    unsigned gpx;
    __device__ __forceinline__ char* rec_ptr(int p) const { return gf + (go_pu + gpx + (((unsigned)p << gsh) * 32u)); }
    __device__ __forceinline__ Blk<T> ldU(int p) const {
        if (kPairRec) { chk_blk(go_pu, p); return ldg_blk(reinterpret_cast<const T*>(rec_ptr(p))); }
        return ldB(so_pu, go_pu, p);
    }
    __device__ __forceinline__ Blk<T> ldL(int p) const {
        if (kPairRec) { chk_blk(go_pu, p); return ldg_blk(reinterpret_cast<const T*>(rec_ptr(p) + 16)); }
        return ldB(so_pl, go_pl, p);
    }
    __device__ __forceinline__ void stU(int p, const Blk<T>& v) const {
        if (kPairRec) { chk_blk(go_pu, p); stg_blk(reinterpret_cast<T*>(rec_ptr(p)), v); }
        else stB(so_pu, go_pu, p, v);
    }
    __device__ __forceinline__ void stL(int p, const Blk<T>& v) const {
        if (kPairRec) { chk_blk(go_pu, p); stg_blk(reinterpret_cast<T*>(rec_ptr(p) + 16), v); }
        else stB(so_pl, go_pl, p, v);
    }
    // both blocks of a pair
    __device__ __forceinline__ void ldUL(int p, Blk<T>& U, Blk<T>& L) const {
        if (kPairRec) {
            chk_blk(go_pu, p);
            float a, b, c, d, e, f, g, h;
            asm volatile("ld.global" SABLE_FAC_LD ".v8.f32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                         : "=f"(a), "=f"(b), "=f"(c), "=f"(d), "=f"(e), "=f"(f), "=f"(g), "=f"(h) : "l"(rec_ptr(p)) : "memory");
            U = {T(a), T(b), T(c), T(d)}; L = {T(e), T(f), T(g), T(h)};
        } else { U = ldU(p); L = ldL(p); }
    }
    __device__ __forceinline__ void stUL(int p, const Blk<T>& U, const Blk<T>& L) const {
        if (kPairRec) {
            chk_blk(go_pu, p);
            asm volatile("st.global" SABLE_FAC_ST ".v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(rec_ptr(p)), "f"(float(U.a)), "f"(float(U.b)), "f"(float(U.c)),
                         "f"(float(U.d)), "f"(float(L.a)), "f"(float(L.b)), "f"(float(L.c)), "f"(float(L.d)) : "memory");
        } else { stU(p, U); stL(p, L); }
    }
    // ask the L2 for the U (h = 0) or L' (h = 1) blocks of the pairs [p0, p1) of this thread's GROUP (HBM workspace; the
    // blocks of a pair range are contiguous across the slots): every lane `tsub` of `nsub` takes every nsub-th 128-byte line
    __device__ __forceinline__ void prefetch_pairs_l2(int p0, int p1, int h, int tsub, int nsub) const {
        if (kP != 2) return;
        const unsigned rec = kPairRec ? 32u : (unsigned)kBlk;
        const char* base = gf - (size_t)(threadIdx.x & ((1 << gsh) - 1)) * kBlk + ((kPairRec || !h) ? go_pu : go_pl);
        const unsigned b0 = (((unsigned)p0 << gsh) * rec) & ~127u, b1 = ((unsigned)p1 << gsh) * rec;
        for (unsigned o = b0 + (unsigned)tsub * 128u; o < b1; o += (unsigned)nsub * 128u)
            asm volatile("prefetch.global.L2 [%0];" ::"l"(base + o));
    }
    // h = 0: the U block of pair p, h = 1: the L' block
    __device__ __forceinline__ Blk<T> ldP(int p, int h) const { return h ? ldL(p) : ldU(p); }
    __device__ __forceinline__ void stP(int p, int h, const Blk<T>& v) const { if (h) stL(p, v); else stU(p, v); }

    __device__ __forceinline__ double2* st_ptr(unsigned so, unsigned go, int m) const {
        chk_st(m);
        if (kP == 0) return reinterpret_cast<double2*>(sb + (so + ((unsigned)m << (gsh + 4))));
        return reinterpret_cast<double2*>(gw + (go + ((unsigned)m << (gsh + 4))));
    }
    __device__ __forceinline__ double2 vv(int m) const { return *st_ptr(0u, 0u, m); }
    __device__ __forceinline__ double2 ma(int m) const { return *st_ptr(so_ma, go_ma, m); }
    __device__ __forceinline__ double2 rh(int m) const { return *st_ptr(so_rh, go_rh, m); }
    __device__ __forceinline__ void set_vv(int m, double2 v) const { *st_ptr(0u, 0u, m) = v; }
    __device__ __forceinline__ void set_ma(int m, double2 v) const { *st_ptr(so_ma, go_ma, m) = v; }
    __device__ __forceinline__ void set_rh(int m, double2 v) const { *st_ptr(so_rh, go_rh, m) = v; }
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

constexpr int kMaxRing = 8;     // ring slots (mbarriers in the shared-memory header)

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
    // a sweep that is not run: its entries still pass through the ring (the producer runs R entries ahead),
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

// A TEAM of `csz` CTAs (one thread-block cluster) can serve one group of scenarios together: every CTA keeps the same
// control state, the targets of a level are dealt over the warps of the whole team, the data lives in the group's HBM slices,
// and the per-level barrier is a cluster barrier with release / acquire semantics (which also drops the L1 lines a peer
// may have made stale).  csz = 1: the CTA works alone and the barrier is __syncthreads.
struct Team { int rank, csz; };
__device__ __forceinline__ int cluster_ctarank() { int r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void team_sync(const Team& tm) {
    if (tm.csz == 1) { __syncthreads(); return; }
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

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
