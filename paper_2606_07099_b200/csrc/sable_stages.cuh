// CTA-wide stage routines of the batched Newton-Raphson power flow (eq. 6-8, eq. 14).  A CTA serves G
// scenario slots in lockstep: thread tid serves slot g = tid % G.  Targets of one elimination level are spread over
// the warps; a target whose multiply-subtract list is long is served by S = 2^s consecutive lane groups that each
// take every S-th term and combine by warp shuffles (lane = (target_in_warp, part, slot), slot fastest).
#pragma once
#include "sable_device.cuh"

namespace sable {

// a1 (+ diagonal case of a2): S = V o conj(Ybus V), F1 rows (eq. 6), real form of
// PAPER.md:201-207; writes rh = -F1 and the diagonal Jacobian blocks (Alg. 1 diagonal case: uses the calculated
// P_i, Q_i -- PAPER.md:193, :215); returns this thread's max |F1| (NaN-propagating).  No barrier, no shuffle.
template <typename T, int kP>
__device__ __forceinline__ double stage_mismatch(const DevTemplate& t, const Slot<T, kP>& s, const double* p_row,
                                                 const double* q_row, bool act, int leaf_m1) {
    // leaf_m1: nodes m < leaf_m1 (level 0: no earlier neighbour, so D_m = J(m,m) and y_m = rhs_m) get their pivot inverse
    // stored right here -- with stage_fill_pairs<kPrescale> and kLeafDone the refactor has nothing left to do at level 0
    // every lane of a warp runs the pass (the row split combines lanes by shuffles); a lane whose slot does not need
    // the evaluation (act = false) takes part in the shuffles and writes nothing
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gsh = s.gsh;
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
            double ire = 0.0, iim = 0.0;
            const int k1 = valid ? row.z : 0;
            for (int k = row.y + part; k < k1; k += S) {
                const int col = t.ycol[k];
                const double2 y = t.ygb[k];
                const double2 x = s.vv(col);
                ire += y.x * x.x - y.y * x.y;
                iim += y.y * x.x + y.x * x.y;
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { ire += shx(ire, o); iim += shx(iim, o); }
            if (lead) {
                const double2 v = s.vv(m);
                const double vm = s.ma(m).x;
                const double P = v.x * ire + v.y * iim, Q = v.y * ire - v.x * iim;
                const bool pq = row.w >> 30;
                const int bus = row.w & kIdxMask;
                const double fp = P - p_row[bus], fq = pq ? Q - q_row[bus] : 0.0;
                s.set_rh(m, make_double2(-fp, -fq));
                loc = nan_max(loc, nan_max(fabs(fp), fabs(fq)));
                const double2 yd = t.ydiag_gb[m];
                const double v2 = vm * vm, iv = 1.0 / vm;
                Blk<T> d;
                d.a = T(-Q - yd.y * v2);
                if (pq) { d.b = T(P * iv + yd.x * vm); d.c = T(P - yd.x * v2); d.d = T(Q * iv - yd.y * vm); }
                else    { d.b = T(0); d.c = T(0); d.d = T(1); }
                s.stD(m, m < leaf_m1 ? inv(d) : d);
            }
        }
    }
    return loc;
}

// a2, off-diagonal case of Alg. 1 (body reconstructed, reading 4) with
// theta_mj = theta_m - theta_j:  a = Vm_m Vm_j cos theta_mj,  b = Vm_m Vm_j sin theta_mj
//   dP_m/dth_j = G b - B a     dP_m/dVm_j = (G a + B b)/Vm_j     dQ_m/dth_j = -(G a + B b)     dQ_m/dVm_j = (G b - B a)/Vm_j
// evaluated in FP64 and rounded to T (Table I: value update DP, solver copy SP).  Fill pairs get zeros.
template <typename T, int kP>
__device__ __forceinline__ void fill_pair(const Slot<T, kP>& s, int2 mj, double4 y, Blk<T>& U, Blk<T>& L) {
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

// a2 as one wide pass over all pairs: every pair slot of the filled pattern is written.  kPrescale: the pairs owned by
// level-0 nodes (p < leaf_p1; such a node has no earlier neighbour, so D_m = J(m,m) and its pairs have no terms) get
// their final values here -- U(m,j) = J(m,j), L(j,m) = J(j,m) J(m,m)^-1 (the inverse comes from stage_mismatch) -- and
// the refactor skips level 0 altogether (kLeafDone).
template <typename T, int kP, bool kPrescale>
__device__ __forceinline__ void stage_fill_pairs(const DevTemplate& t, const Slot<T, kP>& s, int tsub, int nsub, int leaf_p1) {
    for (int p = tsub; p < t.n_pair; p += nsub) {
        Blk<T> U, L;
        const int2 mj = t.pair_mj[p];
        fill_pair<T, kP>(s, mj, t.pair_y[p], U, L);
        if (kPrescale && p < leaf_p1) L = mul(L, s.ldD(mj.x & kIdxMask));       // D^-1 left there by stage_mismatch
        s.stU(p, U); s.stL(p, L);
    }
}

// a4 + forward half of a5: block LU on the static pattern, level by level (unit-lower L, pivot blocks D_m stored
// inverted), fused with the forward substitution L y = rhs which walks the same lists.  Contains barriers.
//   diag target m :  D_m = J(m,m) - sum_k L(m,k) U(k,m);   y_m = rhs_m - sum_k L(m,k) y_k      (k: pairs (k,m))
//   pair target p :  U(m,j) = J(m,j) - sum_k L(m,k) U(k,j);  L(j,m) = (J(j,m) - sum_k L(j,k) U(k,m)) D_m^-1
// kLeafDone: the pairs of level 0 already hold their final values (stage_fill_pairs<kPrescale>), level 0 then has
// diagonal targets only and a single barrier.  A pair target without terms is not touched by the accumulate pass.
// kTransposed runs U^T w = g instead of L y = rhs:  w_m = D_m^-T (g_m - sum_k U(k,m)^T w_k).
// kAll = false: only the levels [0, nl_) are processed (those below the dense top front: sable_front.cuh).
template <typename T, int kP, bool kFactor, bool kSolve, bool kTransposed, bool kLeafDone, bool kAll = true>
__device__ __forceinline__ void stage_factor_forward(const DevTemplate& t, const Slot<T, kP>& s, const LevelDesc* lv, BlobRing& ring, int nl_ = 0) {
    const int nl = kAll ? t.n_level : nl_;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gsh = s.gsh;
    long long tk = clock64();
    for (int l = 0; l < nl; ++l) {
        const LevelDesc d = lv[l];
        const char* lb = ring.acquire(l, d);
        const int* dptr = reinterpret_cast<const int*>(lb);
        const int* tptr = reinterpret_cast<const int*>(lb + d.o_tptr);
        const int2* dak = reinterpret_cast<const int2*>(lb + d.o_dak);
        const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
        const int2* tab = reinterpret_cast<const int2*>(lb + d.o_tab);
        if (!(kLeafDone && l == 0)) {
            const int ssh = d.sd, tsh = 5 - gsh - ssh, S = 1 << ssh;
            const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
            for (int base = d.m0 + (warp << tsh); base < d.m1; base += nwarps << tsh) {
                const bool valid = base + tl < d.m1;
                const int m = valid ? base + tl : d.m1 - 1;
                const bool lead = valid && part == 0;
                const int t0 = dptr[m - d.m0], t1 = valid ? dptr[m - d.m0 + 1] : t0;
                Blk<T> D = {T(0), T(0), T(0), T(0)};
                T y0 = T(0), y1 = T(0);
                if (lead) {
                    if (kFactor) D = s.ldD(m);
                    if (kSolve) { const double2 r = s.rh(m); y0 = T(r.x); y1 = T(r.y); }
                }
                for (int q = t0 + part; q < t1; q += S) {
                    const int2 ak = dak[q];
                    if (kFactor || kTransposed) {
                        const Blk<T> U = s.ldU(ak.x);
                        if (kFactor) mulsub(D, s.ldL(ak.x), U);
                        if (kSolve && kTransposed) { const double2 x = s.rh(ak.y); y0 -= U.a * T(x.x) + U.c * T(x.y);  y1 -= U.b * T(x.x) + U.d * T(x.y); }
                    }
                    if (kSolve && !kTransposed) {
                        const Blk<T> L = s.ldL(ak.x);
                        const double2 x = s.rh(ak.y);
                        y0 -= L.a * T(x.x) + L.b * T(x.y);  y1 -= L.c * T(x.x) + L.d * T(x.y);
                    }
                }
                for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) {
                    if (kFactor) blk_add_shx(D, o);
                    if (kSolve) { y0 += shx(y0, o); y1 += shx(y1, o); }
                }
                if (lead) {
                    if (kFactor) { D = inv(D); s.stD(m, D); }
                    if (kSolve) {
                        if (kTransposed) {
                            if (!kFactor) D = s.ldD(m);
                            const T z0 = D.a * y0 + D.c * y1, z1 = D.b * y0 + D.d * y1; y0 = z0; y1 = z1;
                        }
                        s.set_rh(m, make_double2(double(y0), double(y1)));
                    }
                }
            }
        }
        if (kFactor && !(kLeafDone && l == 0)) {
            // pair targets accumulate J - sum(terms) concurrently with the diagonal targets (they only need factors of
            // earlier levels); warps are taken from the other end so that a narrow level spreads over distinct warps
            const int ssh = d.sp, tsh = 5 - gsh - ssh, S = 1 << ssh;
            const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
            for (int base = d.p0 + ((nwarps - 1 - warp) << tsh); base < d.p1; base += nwarps << tsh) {
                const bool valid = base + tl < d.p1;
                const int p = valid ? base + tl : d.p1 - 1;
                const int t0 = tptr[p - d.p0], t1 = valid ? tptr[p - d.p0 + 1] : t0;
                const bool lead = valid && part == 0 && t1 > t0;
                Blk<T> U = {T(0), T(0), T(0), T(0)}, L = {T(0), T(0), T(0), T(0)};
                if (lead) { U = s.ldU(p); L = s.ldL(p); }
                for (int q = t0 + part; q < t1; q += S) {
                    const int2 ab = tab[q];
                    mulsub(U, s.ldL(ab.x), s.ldU(ab.y));
                    mulsub(L, s.ldL(ab.y), s.ldU(ab.x));
                }
                for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { blk_add_shx(U, o); blk_add_shx(L, o); }
                if (lead) { s.stU(p, U); s.stL(p, L); }
            }
            __syncthreads();
            ring.tick(4 * l, tk);
            // scale: L(j,m) = L'(j,m) D_m^-1 with the pivot inverses of this level
            const int np = d.p1 - d.p0;
            for (int i = threadIdx.x >> gsh; i < np; i += blockDim.x >> gsh) {
                const int p = d.p0 + i;
                s.stL(p, mul(s.ldL(p), s.ldD(pmj[i].x & kIdxMask)));
            }
        }
        if (kLeafDone && l == 0 && !ring.on) continue;   // nothing was done at level 0: no barrier needed
        __syncthreads();
        ring.tick(4 * l + 1, tk);
        ring.release(l);
    }
}

// backward half of a5: U x = y, i.e. x_m = D_m^-1 (y_m - sum_j U(m,j) x_j) over the pairs owned by m, levels
// descending.  kTransposed: L^T lambda = w, lambda_m = w_m - sum_j L(j,m)^T lambda_j.  Contains barriers.
template <typename T, int kP, bool kTransposed, bool kAll = true>
__device__ __forceinline__ void stage_backward(const DevTemplate& t, const Slot<T, kP>& s, const LevelDesc* lv, BlobRing& ring, int nl_ = 0) {
    const int nl = kAll ? t.n_level : nl_;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gsh = s.gsh;
    long long tk = clock64();
    for (int l = nl - 1; l >= 0; --l) {
        const LevelDesc d = lv[l];
        const char* lb = ring.acquire(l, d);
        const int* pptr = reinterpret_cast<const int*>(lb + d.o_pptr);
        const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
        const int ssh = d.sb, tsh = 5 - gsh - ssh, S = 1 << ssh;
        const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
        for (int base = d.m0 + (warp << tsh); base < d.m1; base += nwarps << tsh) {
            const bool valid = base + tl < d.m1;
            const int m = valid ? base + tl : d.m1 - 1;
            const bool lead = valid && part == 0;
            const int p0 = pptr[m - d.m0] & kIdxMask, p1 = valid ? pptr[m - d.m0 + 1] & kIdxMask : p0;
            T y0 = T(0), y1 = T(0);
            if (lead) { const double2 r = s.rh(m); y0 = T(r.x); y1 = T(r.y); }
            for (int pi = p0 + part; pi < p1; pi += S) {
                const int j = pmj[pi].y & kIdxMask, p = d.p0 + pi;
                const double2 x = s.rh(j);
                if (!kTransposed) { const Blk<T> U = s.ldU(p); y0 -= U.a * T(x.x) + U.b * T(x.y); y1 -= U.c * T(x.x) + U.d * T(x.y); }
                else              { const Blk<T> L = s.ldL(p); y0 -= L.a * T(x.x) + L.c * T(x.y); y1 -= L.b * T(x.x) + L.d * T(x.y); }
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { y0 += shx(y0, o); y1 += shx(y1, o); }
            if (lead) {
                if (!kTransposed) {
                    const Blk<T> D = s.ldD(m);
                    const T z0 = D.a * y0 + D.b * y1, z1 = D.c * y0 + D.d * y1; y0 = z0; y1 = z1;
                }
                s.set_rh(m, make_double2(double(y0), double(y1)));
            }
        }
        __syncthreads();
        ring.tick(4 * l + 2, tk);
        ring.release(l);
    }
}

// Newton update of PAPER.md:90 for every node, accumulated in FP64; one wide pass (the sincos is kept
// off the level-by-level critical path of the backward sweep).  No barrier.
template <typename T, int kP>
__device__ __forceinline__ void stage_update(const DevTemplate& t, const Slot<T, kP>& s, int tsub, int nsub) {
    for (int m = tsub; m < t.n_node; m += nsub) {
        const double2 a = s.ma(m), x = s.rh(m);
        const double th = a.y + x.x;
        const double vm = t.node_pq[m] ? a.x + x.y : a.x;
        double sn, cs; sincos(th, &sn, &cs);
        s.set_ma(m, make_double2(vm, th));
        s.set_vv(m, make_double2(vm * cs, vm * sn));
    }
}

}  // namespace sable
