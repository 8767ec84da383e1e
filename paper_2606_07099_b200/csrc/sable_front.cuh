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
//   write-back (kept factors only)  D^-1, U(m,j) = M[r][c], L(j,m) = M[c][r] D_r^-1 into the sparse slots that
//              sable_adjoint's transposed sweeps read.
// Entries outside the static pattern are zero and stay zero (the pattern is closed under fill), so the arithmetic is
// that of the sparse code up to the order of the sums.
#pragma once
#include "sable_device.cuh"

namespace sable {

// bytes of shared memory per CTA: M (K*K blocks), the pivot inverses (K blocks), y (K double2), for 2^gsh slots
template <typename T> __host__ __device__ inline int64_t front_bytes(int K, int gsh) {
    return (((int64_t)K * K + K) * 4 * (int64_t)sizeof(T) + (int64_t)K * 16) << gsh;
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

// Assembly: the accumulate phase of stage_factor_forward for all front targets at once, term lists filtered to sparse
// k (LevelDesc d: m0 = f0, m1 = n_node, p0 .. p1 = the pairs owned by front nodes), results into M and y.  Ends with a
// barrier.  The lead lane of the first front node also leaves D_0^-1.
template <typename T, int kP, bool kSolve>
__device__ __forceinline__ void front_assemble(const DevTemplate& t, const Slot<T, kP>& s, const Front<T>& F, const LevelDesc& d) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5, gsh = s.gsh;
    const char* lb = t.blob + d.blob_off;
    const int* dptr = reinterpret_cast<const int*>(lb);
    const int* tptr = reinterpret_cast<const int*>(lb + d.o_tptr);
    const int2* dak = reinterpret_cast<const int2*>(lb + d.o_dak);
    const int2* pmj = reinterpret_cast<const int2*>(lb + d.o_pmj);
    const int2* tab = reinterpret_cast<const int2*>(lb + d.o_tab);
    {
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
                D = s.ldD(m);
                if (kSolve) { const double2 r = s.rh(m); y0 = T(r.x); y1 = T(r.y); }
            }
            for (int q = t0 + part; q < t1; q += S) {
                const int2 ak = dak[q];
                const Blk<T> L = s.ldL(ak.x);
                mulsub(D, L, s.ldU(ak.x));
                if (kSolve) { const double2 x = s.rh(ak.y); y0 -= L.a * T(x.x) + L.b * T(x.y);  y1 -= L.c * T(x.x) + L.d * T(x.y); }
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) {
                blk_add_shx(D, o);
                if (kSolve) { y0 += shx(y0, o); y1 += shx(y1, o); }
            }
            if (lead) {
                const int r = m - F.f0;
                F.stM(r, r, D);
                if (r == 0) F.stI(0, inv(D));
                if (kSolve) *F.yp(r) = make_double2(double(y0), double(y1));
            }
        }
    }
    {
        const int ssh = d.sp, tsh = 5 - gsh - ssh, S = 1 << ssh;
        const int tl = lane >> (gsh + ssh), part = (lane >> gsh) & (S - 1);
        for (int base = d.p0 + ((nwarps - 1 - warp) << tsh); base < d.p1; base += nwarps << tsh) {
            const bool valid = base + tl < d.p1;
            const int p = valid ? base + tl : d.p1 - 1;
            const int t0 = tptr[p - d.p0], t1 = valid ? tptr[p - d.p0 + 1] : t0;
            const bool lead = valid && part == 0;
            Blk<T> U = {T(0), T(0), T(0), T(0)}, L = {T(0), T(0), T(0), T(0)};
            if (lead) { U = s.ldU(p); L = s.ldL(p); }
            for (int q = t0 + part; q < t1; q += S) {
                const int2 ab = tab[q];
                mulsub(U, s.ldL(ab.x), s.ldU(ab.y));
                mulsub(L, s.ldL(ab.y), s.ldU(ab.x));
            }
            for (int o = (S >> 1) << gsh; o >= (1 << gsh); o >>= 1) { blk_add_shx(U, o); blk_add_shx(L, o); }
            if (lead) {
                const int2 mj = pmj[p - d.p0];
                const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
                F.stM(r, c, U); F.stM(c, r, L);
            }
        }
    }
    __syncthreads();
}

// Right-looking block LU of M with the forward substitution as an extra column.  K barriers.
template <typename T, bool kSolve>
__device__ __forceinline__ void front_factor(const Front<T>& F, int tsub, int nsub) {
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
                    if (i == 0) F.stI(r + 1, inv(X));            // pivot of the next step
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

// kept factors: the front's D^-1, U and scaled L into the sparse slots (pairs p0 .. p1 of LevelDesc d).  No barrier.
template <typename T, int kP>
__device__ __forceinline__ void front_store(const DevTemplate& t, const Slot<T, kP>& s, const Front<T>& F, const LevelDesc& d, int tsub, int nsub) {
    const int2* pmj = reinterpret_cast<const int2*>(t.blob + d.blob_off + d.o_pmj);
    for (int r = tsub; r < F.K; r += nsub) s.stD(F.f0 + r, F.ldI(r));
    for (int i = tsub; i < d.p1 - d.p0; i += nsub) {
        const int2 mj = pmj[i];
        const int r = (mj.x & kIdxMask) - F.f0, c = (mj.y & kIdxMask) - F.f0;
        s.stU(d.p0 + i, F.ldM(r, c));
        s.stL(d.p0 + i, mul(F.ldM(c, r), F.ldI(r)));
    }
}

}  // namespace sable
