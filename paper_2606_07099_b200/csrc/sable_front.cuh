// Dense top front of the elimination tree (fused HBM-placement kernel only).
//
// The last levels of the elimination order hold one or two nodes each whose pattern is (almost) a dense block: on
// the synthetic 9 241-bus grid the last 45 levels are 45 single nodes with 1 000 of the 1 035 possible pairs.  Level by
// level they cost three barrier-separated phases each, every phase a chain of dependent DRAM / L2 round trips, which
// is 40 % of a Newton iteration there.  Here the K front nodes f0 .. n_node-1 (all nodes of the levels >= Lc) are
// treated as ONE dense K x K block matrix M of 2x2 blocks in shared memory:
//   assemble   M = J(front, front) - sum over the SPARSE nodes k < f0 of L(.,k) U(k,.)      (Schur complement; the
//              same pull lists as the level-by-level code, filtered to k < f0: one accumulate phase for the whole front),
//              y_front = rhs_front - sum_k L(.,k) y_k
//   factor     right-looking block LU with the same 2x2 pivots D_r in the same order, one barrier per step:
//              M[c][c'] -= (M[c][r] D_r^-1) M[r][c'],   y_c -= (M[c][r] D_r^-1) y_r        (forward solve fused in)
//   backward   x_c = D_c^-1 y_c;  y_r -= M[r][c] x_c  (r < c),  c descending, one barrier per step
//   write-back (kept factors only)  D^-1, U(m,j) = M[r][c], L'(j,m) = M[c][r] (unscaled, sable_device.cuh) into the sparse
//              slots that sable_adjoint's transposed sweeps read.
// Entries outside the static pattern are zero and stay zero (the pattern is closed under fill), so the arithmetic is
// that of the sparse code up to the order of the sums.
#pragma once
#include "sable_stages.cuh"

namespace sable {

// bytes of shared memory per CTA: M (K*K blocks), the pivot inverses (K blocks), y and w (K double2 each), for 2^gsh slots
template <typename T> __host__ __device__ inline int64_t front_bytes(int K, int gsh) {
    return (((int64_t)K * K + K) * 4 * (int64_t)sizeof(T) + (int64_t)2 * K * 16) << gsh;
}

template <typename T> struct Front {
    static constexpr int VPB = (int)(4 * sizeof(T) / 16);
    char* base;                 // shared memory of this CTA's front, already offset by g * 16
    int K, f0, gsh;
    unsigned o_dinv, o_y;
    __device__ __forceinline__ T* bp(unsigned off, int idx, int& vs) const {
        vs = 16 << gsh; return reinterpret_cast<T*>(base + (off + ((unsigned)(idx * VPB) << (gsh + 4))));
    }
    __device__ __forceinline__ Blk<T> ldM(int r, int c) const { int vs; const T* p = bp(0, r * K + c, vs); return ld_blk(p, vs); }
    __device__ __forceinline__ void stM(int r, int c, const Blk<T>& v) const { int vs; T* p = bp(0, r * K + c, vs); st_blk(p, vs, v); }
    __device__ __forceinline__ Blk<T> ldI(int r) const { int vs; const T* p = bp(o_dinv, r, vs); return ld_blk(p, vs); }
    __device__ __forceinline__ void stI(int r, const Blk<T>& v) const { int vs; T* p = bp(o_dinv, r, vs); st_blk(p, vs, v); }
    __device__ __forceinline__ double2* yp(int r) const { return reinterpret_cast<double2*>(base + (o_y + ((unsigned)r << (gsh + 4)))); }
    __device__ __forceinline__ double2* wp(int r) const { return reinterpret_cast<double2*>(base + (o_y + ((unsigned)(K + r) << (gsh + 4)))); }
};

template <typename T>
__device__ __forceinline__ Front<T> carve_front(unsigned char* smem, int64_t off, int K, int f0, int gsh, int g) {
    Front<T> F;
    F.base = reinterpret_cast<char*>(smem) + off + g * 16; F.K = K; F.f0 = f0; F.gsh = gsh;
    F.o_dinv = (unsigned)(((size_t)K * K * 4 * sizeof(T)) << gsh);
    F.o_y = F.o_dinv + (unsigned)(((size_t)K * 4 * sizeof(T)) << gsh);
    return F;
}

// M = 0 (entries outside the static pattern are never written otherwise).  No barrier.
template <typename T>
__device__ __forceinline__ void front_zero(const Front<T>& F, int tsub, int nsub) {
    const Blk<T> z = {T(0), T(0), T(0), T(0)};
    for (int i = tsub; i < F.K * F.K; i += nsub) { int vs; T* p = F.bp(0, i, vs); st_blk(p, vs, z); }
}

// Assembly: the accumulate phase of a level (accumulate_level, sable_stages.cuh) for all front targets at once, item lists
// filtered to sparse k (LevelDesc d: m0 = f0, m1 = n_node, p0 .. p1 = the pairs owned by front nodes, with its own target
// classes), results into M and y instead of the sparse slots.  The lead lane of the first front node also leaves D_0^-1.
template <typename T> struct FrontSink {
    const Front<T>& F;
    const PivotFlag& pf;
    static constexpr bool kInvert = false;      // pivots are inverted by front_factor, in elimination order
    __device__ __forceinline__ void diag(int m, const Blk<T>& D, T y0, T y1, bool factor, bool solve) const {
        const int r = m - F.f0;
        if (factor) {
            F.stM(r, r, D);
            if (r == 0) { bool bad = false; F.stI(0, inv(D, bad)); if (bad) pf.raise(); }
        }
        if (solve) *F.yp(r) = make_double2(double(y0), double(y1));
    }
    __device__ __forceinline__ void pair(int, int h, int2 mj, const Blk<T>& v) const {
        const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
        if (h) F.stM(c, r, v); else F.stM(r, c, v);
    }
    __device__ __forceinline__ void pair2(int, int2 mj, const Blk<T>& U, const Blk<T>& L) const {
        const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
        F.stM(r, c, U); F.stM(c, r, L);
    }
};

// Fills M and y of the front: entries with terms through accumulate_level, the others straight from the sparse slots
// (where stage_mismatch left J; a fill-in pair without terms below the front stays zero).  Ends with a barrier.
template <typename T, int kP, bool kSolve>
__device__ __forceinline__ void front_assemble(const DevTemplate& t, const Slot<T, kP>& s, const Front<T>& F, const LevelDesc& d,
                                               const PivotFlag& pf, double* scratch, int tsub, int nsub) {
    const char* lb = t.blob + d.blob_off;
    // block-targets without terms (sorted behind the class ranges): copy J(m,j) / J(j,m)
    {
        const int* tord = reinterpret_cast<const int*>(lb + d.o_tord);
        const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
        int with_terms = 0;                         // pair targets with terms: the end of the last pair class
        for (int c = 0; c < d.n_cls; ++c) if (!d.cls[c].diag) with_terms = d.cls[c].i1 / kTargetUnit;
        const int nbt = 2 * (d.p1 - d.p0);
        for (int bt = 2 * with_terms + tsub; bt < nbt; bt += nsub) {
            const int to = tord[bt >> 1], pl = to & kIdxMask, h = bt & 1;
            if (to & kFromZero) continue;
            const int2 mj = pmj[pl];
            const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
            const Blk<T> v = s.ldP(d.p0 + pl, h);
            if (h) F.stM(c, r, v); else F.stM(r, c, v);
        }
    }
    const FrontSink<T> sink{F, pf};
    accumulate_level<T, kP, true, kSolve, false>(s, d, lb, sink, pf, scratch, Team{0, 1});
    __syncthreads();
}

// Right-looking block LU of M with the forward substitution as an extra column.  K barriers.
template <typename T, bool kSolve>
__device__ __forceinline__ void front_factor(const Front<T>& F, const PivotFlag& pf, int tsub, int nsub) {
    const int K = F.K;
    for (int r = 0; r + 1 < K; ++r) {
        const int nr = K - 1 - r, ncol = nr + (kSolve ? 1 : 0), n = nr * ncol;
        if (tsub < n) {
            const Blk<T> Di = F.ldI(r);
            const float rcol = 1.0f / float(ncol);               // i / ncol below is exact for i < 2^20, ncol <= 128
            for (int i = tsub; i < n; i += nsub) {
                const int ci = __float2int_rz((float(i) + 0.5f) * rcol), c = r + 1 + ci, cc = r + 1 + (i - ci * ncol);
                const Blk<T> Lc = mul(F.ldM(c, r), Di);
                if (cc < K) {
                    Blk<T> X = F.ldM(c, cc);
                    mulsub(X, Lc, F.ldM(r, cc));
                    F.stM(c, cc, X);
                    if (i == 0) { bool bad = false; F.stI(r + 1, inv(X, bad)); if (bad) pf.raise(); }   // pivot of the next step
                } else {
                    const double2 yr = *F.yp(r);
                    double2 yc = *F.yp(c);
                    const T a = T(yr.x), b = T(yr.y);
                    yc.x = double(T(yc.x) - (Lc.a * a + Lc.b * b));  yc.y = double(T(yc.y) - (Lc.c * a + Lc.d * b));
                    *F.yp(c) = yc;
                }
            }
        }
        __syncthreads();
    }
}

// U x = y on the front; x goes to rh(f0 + c) of the slot (where the sparse backward sweep and the update read it).
// K barriers.
template <typename T, int kP>
__device__ __forceinline__ void front_backward(const Slot<T, kP>& s, const Front<T>& F, int tsub, int nsub) {
    for (int c = F.K - 1; c >= 0; --c) {
        if (tsub <= c) {
            const Blk<T> Di = F.ldI(c);
            const double2 yc = *F.yp(c);
            const T x0 = Di.a * T(yc.x) + Di.b * T(yc.y), x1 = Di.c * T(yc.x) + Di.d * T(yc.y);
            for (int r = tsub; r <= c; r += nsub) {
                if (r == c) s.set_rh(F.f0 + c, make_double2(double(x0), double(x1)));
                else {
                    const Blk<T> U = F.ldM(r, c);
                    double2 yr = *F.yp(r);
                    yr.x = double(T(yr.x) - (U.a * x0 + U.b * x1));  yr.y = double(T(yr.y) - (U.c * x0 + U.d * x1));
                    *F.yp(r) = yr;
                }
            }
        }
        __syncthreads();
    }
}

// kept factors: the front's D^-1, U and L' into the sparse slots (pairs p0 .. p1 of LevelDesc d).  No barrier.
template <typename T, int kP>
__device__ __forceinline__ void front_store(const DevTemplate& t, const Slot<T, kP>& s, const Front<T>& F, const LevelDesc& d, int tsub, int nsub) {
    const int2* pmj = reinterpret_cast<const int2*>(t.blob + d.blob_off + d.o_pmj);
    for (int r = tsub; r < F.K; r += nsub) s.stD(F.f0 + r, F.ldI(r));
    for (int i = tsub; i < d.p1 - d.p0; i += nsub) {
        const int2 mj = pmj[i];
        const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
        s.stU(d.p0 + i, F.ldM(r, c));
        s.stL(d.p0 + i, F.ldM(c, r));
    }
}

// ---- the front in the adjoint kernel (transposed sweeps on kept factors) ---------------------------------------------
// Load: M[r][c] = U(m,j), M[c][r] = L'(j,m) of the front's pairs and the pivot inverses from the sparse slots (entries
// outside the pattern stay zero: call front_zero and a barrier first).  No barrier.
template <typename T, int kP>
__device__ __forceinline__ void front_load(const DevTemplate& t, const Slot<T, kP>& s, const Front<T>& F, const LevelDesc& d, int tsub, int nsub) {
    const int2* pmj = reinterpret_cast<const int2*>(t.blob + d.blob_off + d.o_pmj);
    for (int r = tsub; r < F.K; r += nsub) F.stI(r, s.ldD(F.f0 + r));
    for (int i = tsub; i < d.p1 - d.p0; i += nsub) {
        const int2 mj = pmj[i];
        const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
        F.stM(r, c, s.ldU(d.p0 + i));
        F.stM(c, r, s.ldL(d.p0 + i));
    }
}

// U^T w = y on the front (y = g - contributions of the sparse nodes, assembled by accumulate_level): ascending,
// w_c = D_c^-T y_c, then y_c' -= U(c,c')^T w_c for c' > c; w goes to F.wp.  K barriers.
template <typename T>
__device__ __forceinline__ void front_forward_t(const Front<T>& F, int tsub, int nsub) {
    for (int c = 0; c < F.K; ++c) {
        if (tsub < F.K - c) {
            const Blk<T> Di = F.ldI(c);
            const double2 yc = *F.yp(c);
            const T w0 = Di.a * T(yc.x) + Di.c * T(yc.y), w1 = Di.b * T(yc.x) + Di.d * T(yc.y);
            for (int e = tsub; e < F.K - c; e += nsub) {
                if (e == 0) *F.wp(c) = make_double2(double(w0), double(w1));
                else {
                    const Blk<T> U = F.ldM(c, c + e);
                    double2 y = *F.yp(c + e);
                    y.x = double(T(y.x) - (U.a * w0 + U.c * w1));  y.y = double(T(y.y) - (U.b * w0 + U.d * w1));
                    *F.yp(c + e) = y;
                }
            }
        }
        __syncthreads();
    }
}

// (L' D^-1)^T lambda = w on the front: descending, lambda_j = w_j - D_j^-T acc_j, then acc_c += L'(j,c)^T lambda_j for c < j;
// lambda goes to rh(f0 + j) of the slot.  acc lives in F.yp (zeroed here).  K + 1 barriers.
template <typename T, int kP>
__device__ __forceinline__ void front_backward_t(const Slot<T, kP>& s, const Front<T>& F, int tsub, int nsub) {
    for (int r = tsub; r < F.K; r += nsub) *F.yp(r) = make_double2(0.0, 0.0);
    __syncthreads();
    for (int j = F.K - 1; j >= 0; --j) {
        if (tsub <= j) {
            const Blk<T> Di = F.ldI(j);
            const double2 a = *F.yp(j), w = *F.wp(j);
            const T l0 = T(w.x) - (Di.a * T(a.x) + Di.c * T(a.y)), l1 = T(w.y) - (Di.b * T(a.x) + Di.d * T(a.y));
            for (int c = tsub; c <= j; c += nsub) {
                if (c == j) s.set_rh(F.f0 + j, make_double2(double(l0), double(l1)));
                else {
                    const Blk<T> L = F.ldM(j, c);
                    double2 y = *F.yp(c);
                    y.x = double(T(y.x) + (L.a * l0 + L.c * l1));  y.y = double(T(y.y) + (L.b * l0 + L.d * l1));
                    *F.yp(c) = y;
                }
            }
        }
        __syncthreads();
    }
}

}  // namespace sable
