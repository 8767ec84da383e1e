// CTA-wide stage routines of the batched Newton-Raphson power flow (eq. 6-8, eq. 14).  A CTA serves G
// scenario slots in lockstep: thread tid serves slot g = tid % G.  Targets of one elimination level are spread over
// the warps; a target whose multiply-subtract list is long is served by S = 2^s consecutive lane groups that each
// take every S-th item and combine by warp shuffles (lane = (target_in_warp, part, slot), slot fastest).  The targets
// of a level are sorted by list length and cut into classes with their own S (LevelDesc::dcls / tcls); the few
// diagonal targets with very long lists ("big": hubs with hundreds of eliminated neighbours) are served by every warp
// of the CTA in turn, combined through shared memory.
#pragma once
#include "sable_device.cuh"

namespace sable {

#ifndef SABLE_MM_UNROLL
#define SABLE_MM_UNROLL 3
#endif
// Where the off-diagonal Jacobian blocks are evaluated: inside the mismatch walk (one block per Y entry, no second pass over
// the state), or -- FP32 pair records, where a lane must write both blocks of a pair at once -- in a pass over the pairs
#ifndef SABLE_WALK_FILL
#define SABLE_WALK_FILL 1
#endif
template <typename T, int kP> struct FillMode {
    static constexpr bool kWalk = SABLE_WALK_FILL && kP == 2 && !Slot<T, kP>::kPairRec;   // measured: the walk form pays in the HBM workspace with FP64 blocks only
    static constexpr int kUnroll = kWalk ? SABLE_MM_UNROLL : 4;                            // Y entries per step and lane
};

#ifndef SABLE_BWD_PREFETCH
#define SABLE_BWD_PREFETCH 1
#endif
#ifndef SABLE_BWD_AHEAD
#define SABLE_BWD_AHEAD 2
#endif
constexpr int kBwdAhead = SABLE_BWD_AHEAD;
constexpr int kBwdPrefetchPairs = 512;      // levels with more pairs than this are throughput-bound: no prefetch

// Per-thread handle for reporting a tiny pivot: points at the scenario's flag word, or at
// nothing for lanes that serve no scenario.
struct PivotFlag {
    int32_t* w;
    __device__ __forceinline__ void raise() const { if (w) atomicOr(w, 3); }
};

// a1 + a2 in one walk over the Y rows: S = V o conj(Ybus V), F1 rows (eq. 6), real form of
// PAPER.md:201-207; writes rh = -F1, the diagonal Jacobian blocks (Alg. 1 diagonal case: uses the calculated P_i, Q_i --
// PAPER.md:193, :215) and, entry by entry, the off-diagonal blocks (Alg. 1 off-diagonal case; body
// reconstructed, reading 4): with t = Y_mj V_j (the term the row sum needs anyway) and V_m conj(t) = u2 + i u1,
//   u2 = Vm_m Vm_j (G cos th_mj + B sin th_mj),   u1 = Vm_m Vm_j (G sin th_mj - B cos th_mj)
//   dP_m/dth_j = u1     dP_m/dVm_j = u2 / Vm_j     dQ_m/dth_j = -u2     dQ_m/dVm_j = u1 / Vm_j
// evaluated in FP64 and rounded to T (Table I: value update DP, solver copy SP); rows / columns of the identity
// padding of PV nodes are zero.  The block goes to the U half (j later than m in the elimination order) or the L' half of
// its pair; fill-in pairs have no entry and are not written (their targets start from zero: kFromZero).  Returns this
// thread's max |F1| (NaN-propagating).  No barrier, no shuffle beyond the row split.
template <typename T, int kP>
__device__ __forceinline__ double stage_mismatch(const DevTemplate& t, const Slot<T, kP>& s, const double* p_row,
                                                 const double* q_row, bool act, int leaf_m1, const PivotFlag& pf, const Team& tm) {
    // leaf_m1: nodes m < leaf_m1 (level 0: no earlier neighbour, so D_m = J(m,m) and y_m = rhs_m) get their pivot inverse
    // and z_m = D_m^-1 rhs_m stored right here -- the refactor then has nothing to do at level 0 (kLeafDone)
    // every lane of a warp runs the pass (the row split combines lanes by shuffles); a lane whose slot does not need
    // the evaluation (act = false) takes part in the shuffles; its slot is bound to the spare workspace group
    constexpr bool kWalk = FillMode<T, kP>::kWalk;
    constexpr int kU = FillMode<T, kP>::kUnroll;
    const int lane = threadIdx.x & 31, nwarps = (blockDim.x >> 5) * tm.csz, warp = tm.rank * (blockDim.x >> 5) + (threadIdx.x >> 5), gsh = s.gsh;
    double loc = 0.0;
    for (int c = 0; c < t.n_class; ++c) {
        const RowClass rc = t.mm_class[c];
        const int ssh = min(rc.ssh, 5 - gsh), tsh = 5 - gsh - ssh, S = 1 << ssh;
        const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
        for (int base = rc.i0 + (warp << tsh); base < rc.i1; base += nwarps << tsh) {
            const bool valid = base + tl < rc.i1;
            const int4 row = t.mm_row[valid ? base + tl : rc.i1 - 1];
            const int m = row.x;
            const bool lead = valid && part == 0 && act;
            const bool pq = row.w >> 30;
            double2 v = make_double2(0.0, 0.0);
            if (kWalk) v = s.vv(m);
            double ire = 0.0, iim = 0.0;
            const int k1 = valid ? row.z : 0;
            // kU entries per step: their index / admittance loads are issued together, then the V gathers -- a lane
            // that walks a row alone has 2 dependent round trips per step instead of 2 per entry
            for (int k = row.y + part; k < k1; k += kU * S) {
                int2 cd[kU]; double2 y[kU], x[kU];
#pragma unroll
                for (int u = 0; u < kU; ++u) {
                    const int ku = k + u * S;
                    const bool on = ku < k1;
                    if (kWalk) cd[u] = on ? t.ycd[ku] : make_int2(m, -1);
                    else cd[u] = make_int2(on ? t.ycol[ku] : m, -1);
                    y[u] = on ? t.ygb[ku] : make_double2(0.0, 0.0);
                }
#pragma unroll
                for (int u = 0; u < kU; ++u) x[u] = s.vv(cd[u].x);
#pragma unroll
                for (int u = 0; u < kU; ++u) {
                    if (!kWalk) {
                        ire += y[u].x * x[u].x - y[u].y * x[u].y;
                        iim += y[u].y * x[u].x + y[u].x * x[u].y;
                        continue;
                    }
                    const double tr = y[u].x * x[u].x - y[u].y * x[u].y, ti = y[u].y * x[u].x + y[u].x * x[u].y;
                    ire += tr; iim += ti;
                    if (cd[u].y >= 0) {
                        const double u2 = v.x * tr + v.y * ti, u1 = v.y * tr - v.x * ti;
                        const double iv = (cd[u].y >> 30) ? rsqrt(x[u].x * x[u].x + x[u].y * x[u].y) : 0.0;
                        Blk<T> J;
                        J.a = T(u1);  J.b = T(u2 * iv);  J.c = pq ? T(-u2) : T(0);  J.d = pq ? T(u1 * iv) : T(0);
                        s.stP(cd[u].y & kPairMask, (cd[u].y >> 29) & 1, J);
                    }
                }
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { ire += shx(ire, o); iim += shx(iim, o); }
            if (lead) {
                if (!kWalk) v = s.vv(m);
                const double vm = s.ma(m).x;
                const double P = v.x * ire + v.y * iim, Q = v.y * ire - v.x * iim;
                const int bus = row.w & kIdxMask;
                const double fp = P - p_row[bus], fq = pq ? Q - q_row[bus] : 0.0;
                loc = nan_max(loc, nan_max(fabs(fp), fabs(fq)));
                const double2 yd = t.ydiag_gb[m];
                const double v2 = vm * vm, iv = 1.0 / vm;
                Blk<T> d;
                d.a = T(-Q - yd.y * v2);
                if (pq) { d.b = T(P * iv + yd.x * vm); d.c = T(P - yd.x * v2); d.d = T(Q * iv - yd.y * vm); }
                else    { d.b = T(0); d.c = T(0); d.d = T(1); }
                if (m < leaf_m1) {
                    bool bad = false;
                    const Blk<T> di = inv(d, bad);
                    if (bad) pf.raise();
                    s.stD(m, di);
                    const T r0 = T(-fp), r1 = T(-fq);
                    s.set_rh(m, make_double2(double(di.a * r0 + di.b * r1), double(di.c * r0 + di.d * r1)));
                } else {
                    s.stD(m, d);
                    s.set_rh(m, make_double2(-fp, -fq));
                }
            }
        }
    }
    return loc;
}

// a2 as a pass over the pairs that have a Y entry (FillMode::kWalk = false), same blocks as the walk above:
// a = Vm_m Vm_j cos theta_mj, b = Vm_m Vm_j sin theta_mj; both blocks of a pair leave in one store.
template <typename T, int kP>
__device__ __forceinline__ void fill_pair(const Slot<T, kP>& s, int4 mj, double4 y, Blk<T>& U, Blk<T>& L) {
    const int m = mj.x & kIdxMask, j = mj.y & kIdxMask;
    const bool mpq = mj.x >> 30, jpq = mj.y >> 30;
    const double2 vm_ = s.vv(m), vj = s.vv(j);
    const double a = vm_.x * vj.x + vm_.y * vj.y, b = vm_.y * vj.x - vm_.x * vj.y;
    const double ivm = mpq ? 1.0 / s.ma(m).x : 0.0, ivj = jpq ? 1.0 / s.ma(j).x : 0.0;
    const double u1 = y.x * b - y.y * a, u2 = y.x * a + y.y * b;        // block (m,j), Y_mj
    const double l1 = -y.z * b - y.w * a, l2 = y.z * a - y.w * b;       // block (j,m), Y_jm, theta_jm = -theta_mj
    U.a = T(u1);  U.b = T(u2 * ivj);  U.c = mpq ? T(-u2) : T(0);  U.d = mpq ? T(u1 * ivj) : T(0);
    L.a = T(l1);  L.b = T(l2 * ivm);  L.c = jpq ? T(-l2) : T(0);  L.d = jpq ? T(l1 * ivm) : T(0);
}
template <typename T, int kP>
__device__ __forceinline__ void stage_fill_pairs(const DevTemplate& t, const Slot<T, kP>& s, int tsub, int nsub) {
    if (FillMode<T, kP>::kWalk) return;
    // two pairs per step and lane: the index / admittance loads of both are issued before the state gathers of either
    for (int i = tsub; i < t.n_jpair; i += 2 * nsub) {
        const int i2 = i + nsub;
        const bool on2 = i2 < t.n_jpair;
        const int4 mj0 = t.jp_mj[i], mj1 = t.jp_mj[on2 ? i2 : i];
        const double4 y0 = t.jp_y[i], y1 = t.jp_y[on2 ? i2 : i];
        Blk<T> U0, L0, U1, L1;
        fill_pair<T, kP>(s, mj0, y0, U0, L0);
        fill_pair<T, kP>(s, mj1, y1, U1, L1);
        s.stUL(mj0.z, U0, L0);
        if (on2) s.stUL(mj1.z, U1, L1);
    }
}

// Where the accumulate phase of a level leaves its results: the sparse slots (stage_factor_forward) or the dense top
// front in shared memory (front_assemble, sable_front.cuh).
template <typename T, int kP> struct SparseSink {
    const Slot<T, kP>& s;
    static constexpr bool kInvert = true;       // the lead lane inverts the pivot block and applies it to y
    __device__ __forceinline__ void diag(int m, const Blk<T>& Dinv, T z0, T z1, bool factor, bool solve) const {
        if (factor) s.stD(m, Dinv);
        if (solve) s.set_rh(m, make_double2(double(z0), double(z1)));
    }
    __device__ __forceinline__ void pair(int p, int h, int2, const Blk<T>& v) const { s.stP(p, h, v); }
    __device__ __forceinline__ void pair2(int p, int2, const Blk<T>& U, const Blk<T>& L) const { s.stUL(p, U, L); }
};

// Accumulate phase of one level (or of the front's assembly), the heart of a4 + the forward half of a5.  With the
// factorisation J1 = L' D^-1 U (sable_device.cuh):
//   diag target m :  D_m = J(m,m) - sum_a L'(a) D_k^-1 U(a);   y_m = rhs_m - sum_a L'(a) z_k;   z_m = D_m^-1 y_m     (a = pair (k,m))
//   block-target  :  U(m,j) = J(m,j) - sum L'(a) D_k^-1 U(b)   (h = 0);   L'(j,m) = J(j,m) - sum L'(b) D_k^-1 U(a)   (h = 1)
// kTransposed (solve only) runs U^T w = g instead:  w_m = D_m^-T (g_m - sum_a U(a)^T w_k).
// No barrier except around the big targets (d.n_big > 0), whose partial sums go through `scratch` (kBigScratch bytes per slot).
constexpr int kBigDoubles = 6;      // D (4) + y (2) per warp partial
template <typename T, int kP, bool kFactor, bool kSolve, bool kTransposed, typename Sink>
__device__ __forceinline__ void accumulate_level(const Slot<T, kP>& s, const LevelDesc& d, const char* lb, const Sink& sink,
                                                 const PivotFlag& pf, double* scratch, const Team& tm) {
    // warps of the whole team; the big targets (CTA-wide through this CTA's shared memory) only when the CTA works alone
    const int lane = threadIdx.x & 31, nwarps = (blockDim.x >> 5) * tm.csz, warp = tm.rank * (blockDim.x >> 5) + (threadIdx.x >> 5), gsh = s.gsh, G = 1 << gsh;
    const int* dptr = reinterpret_cast<const int*>(lb);
    const int* dord = reinterpret_cast<const int*>(lb + d.o_dord);
    const int2* dak = reinterpret_cast<const int2*>(lb + d.o_dak);
    auto diag_item = [&](const int2 ak, Blk<T>& D, T& y0, T& y1) {
        Blk<T> U, L;
        if (kFactor) s.ldUL(ak.x, U, L);                    // both blocks of the pair (one access with FP32 factors)
        else if (kTransposed) U = s.ldU(ak.x);
        else L = s.ldL(ak.x);
        if (kFactor) mulsub(D, mul(L, s.ldD(ak.y)), U);
        if (kSolve && kTransposed) { const double2 x = s.rh(ak.y); y0 -= U.a * T(x.x) + U.c * T(x.y);  y1 -= U.b * T(x.x) + U.d * T(x.y); }
        if (kSolve && !kTransposed) {
            const double2 x = s.rh(ak.y);
            y0 -= L.a * T(x.x) + L.b * T(x.y);  y1 -= L.c * T(x.x) + L.d * T(x.y);
        }
    };
    // (solve-only sweeps: D holds the kept pivot inverse, loaded by the caller before the item loop)
    auto diag_finish = [&](int m, Blk<T> D, T y0, T y1) {
        Blk<T> Di = D;
        if (Sink::kInvert) {
            if (kFactor) { bool bad = false; Di = inv(D, bad); if (bad) pf.raise(); }
            if (kSolve) {
                const T z0 = kTransposed ? Di.a * y0 + Di.c * y1 : Di.a * y0 + Di.b * y1;
                const T z1 = kTransposed ? Di.b * y0 + Di.d * y1 : Di.c * y0 + Di.d * y1;
                y0 = z0; y1 = z1;
            }
        }
        sink.diag(m, Di, y0, y1, kFactor, kSolve);
    };
    // ---- big diagonal targets: one at a time, every lane of the CTA takes every (lanes)-th item ----------------------
    for (int i = 0; i < (tm.csz == 1 ? d.n_big : 0); ++i) {
        const int m = d.m0 + dord[i], t0 = dptr[i], t1 = dptr[i + 1];
        Blk<T> D = {T(0), T(0), T(0), T(0)};
        T y0 = T(0), y1 = T(0);
        for (int q = t0 + (threadIdx.x >> gsh); q < t1; q += blockDim.x >> gsh) diag_item(dak[q], D, y0, y1);
        for (int o = 16; o >= G; o >>= 1) {
            if (kFactor) blk_add_shx(D, o);
            if (kSolve) { y0 += shx(y0, o); y1 += shx(y1, o); }
        }
        __syncthreads();                                   // scratch free (previous big target consumed)
        if (lane < G) {
            double* w = scratch + ((size_t)(threadIdx.x >> 5) * G + lane) * kBigDoubles;
            w[0] = double(D.a); w[1] = double(D.b); w[2] = double(D.c); w[3] = double(D.d); w[4] = double(y0); w[5] = double(y1);
        }
        __syncthreads();
        if (threadIdx.x < G) {
            double a[kBigDoubles] = {0, 0, 0, 0, 0, 0};
            for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
#pragma unroll
                for (int e = 0; e < kBigDoubles; ++e) a[e] += scratch[((size_t)w * G + threadIdx.x) * kBigDoubles + e];
            }
            Blk<T> Dm = {T(0), T(0), T(0), T(0)};
            T r0 = T(0), r1 = T(0);
            if (kFactor) { const Blk<T> J = s.ldD(m); Dm = {J.a + T(a[0]), J.b + T(a[1]), J.c + T(a[2]), J.d + T(a[3])}; }
            else if (Sink::kInvert) Dm = s.ldD(m);
            if (kSolve) { const double2 r = s.rh(m); r0 = T(r.x) + T(a[4]); r1 = T(r.y) + T(a[5]); }
            diag_finish(m, Dm, r0, r1);
        }
    }
    // ---- tasks: a warp-sized group of targets of one class; dealt to the warps round-robin ---------------------------
    const int* tptr = reinterpret_cast<const int*>(lb + d.o_tptr);
    const int* tord = reinterpret_cast<const int*>(lb + d.o_tord);
    const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
    const int4* tab = reinterpret_cast<const int4*>(lb + d.o_tab);
    const int ncls = d.n_cls;
    int c = 0, tc0 = 0, tc1 = 0;                           // class of the current task and its task range [tc0, tc1)
    auto class_tasks = [&](int cc) { const Cls k = d.cls[cc]; const int tsh = 5 - gsh - min((int)k.ssh, 5 - gsh); return ((k.i1 - k.start) + (1 << tsh) - 1) >> tsh; };
    if (ncls > 0) tc1 = class_tasks(0);
    for (int t = warp; ; t += nwarps) {
        while (c < ncls && t >= tc1) { ++c; tc0 = tc1; if (c < ncls) tc1 += class_tasks(c); }
        if (c >= ncls) break;
        const Cls k = d.cls[c];
        if (!kFactor && !k.diag) break;                    // solve-only sweeps have no pair targets (diagonal classes come first)
        const int ssh = min((int)k.ssh, 5 - gsh), tsh = 5 - gsh - ssh, S = 1 << ssh;
        const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
        const int idx = k.start + ((t - tc0) << tsh) + tl;
        const bool valid = idx < k.i1, lead = valid && part == 0;
        const int i = valid ? idx : k.i1 - 1;
        if (k.diag) {
            const int m = d.m0 + dord[i];
            const int t0 = dptr[i], t1 = valid ? dptr[i + 1] : t0;
            Blk<T> D = {T(0), T(0), T(0), T(0)};
            T y0 = T(0), y1 = T(0);
            if (lead) {
                if (kFactor || Sink::kInvert) D = s.ldD(m);   // J(m,m), or (solve-only) the kept pivot inverse
                if (kSolve) { const double2 r = s.rh(m); y0 = T(r.x); y1 = T(r.y); }
            }
            for (int q = t0 + part; q < t1; q += S) diag_item(dak[q], D, y0, y1);
            for (int o = (S >> 1) << gsh; o >= G; o >>= 1) {
                if (kFactor) blk_add_shx(D, o);
                if (kSolve) { y0 += shx(y0, o); y1 += shx(y1, o); }
            }
            if (lead) diag_finish(m, D, y0, y1);
        } else if (kFactor) {
#if SABLE_HALF_TARGETS
            // block-targets bt = 2 i + h (h = 0: U(m,j), h = 1: L'(j,m)): one uniform item acc -= A D_k^-1 B, three operand blocks
            const int ip = i >> 1, h = i & 1;
            const int t0 = tptr[ip], t1 = valid ? tptr[ip + 1] : t0;
            const int to = tord[ip], pl = to & kIdxMask, p = d.p0 + pl;
            Blk<T> acc = {T(0), T(0), T(0), T(0)};
            if (lead && !(to & kFromZero)) acc = s.ldP(p, h);
            for (int q = t0 + part; q < t1; q += S) {
                const int4 ab = tab[q];
                const Blk<T> W = mul(s.ldL(h ? ab.y : ab.x), s.ldD(ab.z));
                mulsub(acc, W, s.ldU(h ? ab.x : ab.y));
            }
            for (int o = (S >> 1) << gsh; o >= G; o >>= 1) blk_add_shx(acc, o);
            if (lead) sink.pair(p, h, pmj[pl], acc);
#else
            // whole pair targets: five operand blocks in flight per item, both accumulators in one lane
            const int t0 = tptr[i], t1 = valid ? tptr[i + 1] : t0;
            const int to = tord[i], pl = to & kIdxMask, p = d.p0 + pl;
            Blk<T> U = {T(0), T(0), T(0), T(0)}, L = {T(0), T(0), T(0), T(0)};
            if (lead && !(to & kFromZero)) s.ldUL(p, U, L);
            for (int q = t0 + part; q < t1; q += S) {
                const int4 ab = tab[q];
                const Blk<T> Dk = s.ldD(ab.z);
                Blk<T> La, Ua, Lb, Ub;
                s.ldUL(ab.x, Ua, La); s.ldUL(ab.y, Ub, Lb);
                mulsub(U, mul(La, Dk), Ub);
                mulsub(L, mul(Lb, Dk), Ua);
            }
            for (int o = (S >> 1) << gsh; o >= G; o >>= 1) { blk_add_shx(U, o); blk_add_shx(L, o); }
            if (lead) sink.pair2(p, pmj[pl], U, L);
#endif
        }
    }
}

// a4 + forward half of a5 level by level.  One barrier per level.  kLeafDone: level 0 needs nothing (stage_mismatch left
// D^-1 and z of its nodes and the final values of its pairs).  kAll = false: only the levels [0, nl_) are
// processed (those below the dense top front: sable_front.cuh).
template <typename T, int kP, bool kFactor, bool kSolve, bool kTransposed, bool kLeafDone, bool kAll = true>
__device__ __forceinline__ void stage_factor_forward(const DevTemplate& t, const Slot<T, kP>& s, const LevelDesc* lv, BlobRing& ring,
                                                     const PivotFlag& pf, double* scratch, const Team& tm, int nl_ = 0) {
    const int nl = kAll ? t.n_level : nl_;
    long long tk = clock64();
    const SparseSink<T, kP> sink{s};
    for (int l = 0; l < nl; ++l) {
        const LevelDesc& d = lv[l];
        const char* lb = ring.acquire(l, d);
        if (!(kLeafDone && l == 0)) accumulate_level<T, kP, kFactor, kSolve, kTransposed>(s, d, lb, sink, pf, scratch, tm);
        if (kLeafDone && l == 0 && !ring.on) continue;   // nothing was done at level 0: no barrier needed
        team_sync(tm);
        ring.tick(4 * l, tk);
        ring.release(l);
    }
}

// backward half of a5: U x = y with rh holding z = D^-1 y, i.e. x_m = z_m - D_m^-1 sum_j U(m,j) x_j over the pairs owned
// by m, levels descending.  kTransposed: (L' D^-1)^T lambda = w, lambda_m = w_m - D_m^-T sum_j L'(j,m)^T lambda_j.
// Contains barriers.
template <typename T, int kP, bool kTransposed, bool kAll = true>
__device__ __forceinline__ void stage_backward(const DevTemplate& t, const Slot<T, kP>& s, const LevelDesc* lv, BlobRing& ring, const Team& tm, int nl_ = 0) {
    const int nl = kAll ? t.n_level : nl_;
    const int lane = threadIdx.x & 31, nwarps = (blockDim.x >> 5) * tm.csz, warp = tm.rank * (blockDim.x >> 5) + (threadIdx.x >> 5), gsh = s.gsh;
    long long tk = clock64();
    for (int l = nl - 1; l >= 0; --l) {
        const LevelDesc& d = lv[l];
        const char* lb = ring.acquire(l, d);
        const int* pptr = reinterpret_cast<const int*>(lb + d.o_pptr);
        const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
#if SABLE_BWD_PREFETCH
        // the next level's blocks (one contiguous pair range) on their way into the L2 while this level's chain runs
        for (int a = (l == nl - 1 ? 1 : kBwdAhead); a <= kBwdAhead; ++a)
            if (l - a >= 0 && lv[l - a].p1 - lv[l - a].p0 <= kBwdPrefetchPairs)
                s.prefetch_pairs_l2(lv[l - a].p0, lv[l - a].p1, kTransposed ? 1 : 0, threadIdx.x >> gsh, blockDim.x >> gsh);
#endif
        const int ssh = min((int)d.sb, 5 - gsh), tsh = 5 - gsh - ssh, S = 1 << ssh;
        const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
        for (int base = d.m0 + (warp << tsh); base < d.m1; base += nwarps << tsh) {
            const bool valid = base + tl < d.m1;
            const int m = valid ? base + tl : d.m1 - 1;
            const bool lead = valid && part == 0;
            const int p0 = pptr[m - d.m0], p1 = valid ? pptr[m - d.m0 + 1] : p0;
            T y0 = T(0), y1 = T(0);
            // the lead lane's own pivot inverse and right-hand side: asked for before the pair loop, not after the reduction
            // (one dependent memory round trip less per level)
            const bool fin = lead && p1 > p0;
            Blk<T> D = {T(0), T(0), T(0), T(0)};
            double2 r = make_double2(0.0, 0.0);
            if (fin) { D = s.ldD(m); r = s.rh(m); }
            for (int pi = p0 + part; pi < p1; pi += S) {
                const int j = pmj[pi].y & kIdxMask, p = d.p0 + pi;
                const double2 x = s.rh(j);
                if (!kTransposed) { const Blk<T> U = s.ldU(p); y0 += U.a * T(x.x) + U.b * T(x.y); y1 += U.c * T(x.x) + U.d * T(x.y); }
                else              { const Blk<T> L = s.ldL(p); y0 += L.a * T(x.x) + L.c * T(x.y); y1 += L.b * T(x.x) + L.d * T(x.y); }
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { y0 += shx(y0, o); y1 += shx(y1, o); }
            if (fin) {
                const T z0 = kTransposed ? D.a * y0 + D.c * y1 : D.a * y0 + D.b * y1;
                const T z1 = kTransposed ? D.b * y0 + D.d * y1 : D.c * y0 + D.d * y1;
                s.set_rh(m, make_double2(double(T(r.x) - z0), double(T(r.y) - z1)));
            }
        }
        team_sync(tm);
        ring.tick(4 * l + 2, tk);
        ring.release(l);
    }
}

// Newton update of PAPER.md:90 for every node, accumulated in FP64; one wide pass (the sincos is kept
// off the level-by-level critical path of the backward sweep).  No barrier.
template <typename T, int kP>
__device__ __forceinline__ void stage_update(const DevTemplate& t, const Slot<T, kP>& s, int tsub, int nsub) {
    for (int m = tsub; m < t.n_node; m += 2 * nsub) {
        const int m2 = m + nsub < t.n_node ? m + nsub : m;
        const double2 a0 = s.ma(m), x0 = s.rh(m), a1 = s.ma(m2), x1 = s.rh(m2);
        const bool q0 = t.node_pq[m], q1 = t.node_pq[m2];
        const double th0 = a0.y + x0.x, th1 = a1.y + x1.x;
        const double vm0 = q0 ? a0.x + x0.y : a0.x, vm1 = q1 ? a1.x + x1.y : a1.x;
        double sn0, cs0, sn1, cs1; sincos(th0, &sn0, &cs0); sincos(th1, &sn1, &cs1);
        s.set_ma(m, make_double2(vm0, th0));
        s.set_vv(m, make_double2(vm0 * cs0, vm0 * sn0));
        if (m2 != m) {
            s.set_ma(m2, make_double2(vm1, th1));
            s.set_vv(m2, make_double2(vm1 * cs1, vm1 * sn1));
        }
    }
}

}  // namespace sable
