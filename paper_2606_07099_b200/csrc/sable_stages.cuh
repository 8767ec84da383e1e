// Per-scenario stage routines (one CTA = one scenario).  See sable_device.cuh for the block conventions.
#pragma once
#include "sable_device.cuh"

namespace sable {

// Per-scenario working set.  Pointers are generic: they point into shared memory or into the scenario's slice of
// the HBM workspace, depending on the placement chosen at sable_create (sable_info.placement).
template <typename T> struct Scen {
    double *vre, *vim, *vmag, *ang;   // [n_node+1] node order, entry n_node = slack
    double *psp, *qsp;                // [n_node]   specified injections in node order
    double *rhs;                      // [2*n_node] -F, then y, then dz (or g, w, lambda for the adjoint)
    T *dg, *pr;                       // factors
};

// a1 (+ diagonal part of a2): S = V o conj(Ybus V), F1 rows (eq. 6), real form of
// PAPER.md:201-207; writes rhs = -F1, the diagonal Jacobian blocks (Alg. 1 diagonal case: uses the calculated
// P_i, Q_i -- PAPER.md:193, :215) and returns this thread's max |F1| (NaN-propagating).  Reads vre/vim/vmag.
template <typename T>
__device__ __forceinline__ double stage_mismatch(const DevTemplate& t, const Scen<T>& s, bool write_diag) {
    double loc = 0.0;
    for (int m = threadIdx.x; m < t.n_node; m += blockDim.x) {
        double ire = 0.0, iim = 0.0;
        const int k1 = t.yptr[m + 1];
        for (int k = t.yptr[m]; k < k1; ++k) {
            const int c = t.ycol[k];
            const double2 y = t.ygb[k];
            const double xr = s.vre[c], xi = s.vim[c];
            ire += y.x * xr - y.y * xi;
            iim += y.y * xr + y.x * xi;
        }
        const double vr = s.vre[m], vi = s.vim[m], vm = s.vmag[m];
        const double P = vr * ire + vi * iim, Q = vi * ire - vr * iim;
        const bool pq = t.node_pq[m];
        const double fp = P - s.psp[m], fq = pq ? Q - s.qsp[m] : 0.0;
        s.rhs[2 * m] = -fp;
        s.rhs[2 * m + 1] = -fq;
        const double ap = fabs(fp), aq = fabs(fq);
        if (!(ap <= loc)) loc = (ap != ap || loc != loc) ? ap + loc : ap;
        if (!(aq <= loc)) loc = (aq != aq || loc != loc) ? aq + loc : aq;
        if (write_diag) {
            const double2 yd = t.ydiag_gb[m];
            const double v2 = vm * vm;
            Blk<T> d;
            d.a = T(-Q - yd.y * v2);
            if (pq) { d.b = T(P / vm + yd.x * vm); d.c = T(P - yd.x * v2); d.d = T(Q / vm - yd.y * vm); }
            else    { d.b = T(0); d.c = T(0); d.d = T(1); }
            st_blk(s.dg + 4 * m, d);
        }
    }
    return loc;
}

// a2, off-diagonal case of Alg. 1 (body reconstructed, reading 4) with
// theta_mj = theta_m - theta_j:  a = Vm_m Vm_j cos theta_mj,  b = Vm_m Vm_j sin theta_mj
//   dP_m/dth_j = G b - B a     dP_m/dVm_j = (G a + B b)/Vm_j     dQ_m/dth_j = -(G a + B b)     dQ_m/dVm_j = (G b - B a)/Vm_j
// Every pair slot of the filled pattern is written (fill pairs get zeros) so refactor starts from a ready array.
template <typename T>
__device__ __forceinline__ void stage_fill_pairs(const DevTemplate& t, const Scen<T>& s) {
    for (int p = threadIdx.x; p < t.n_pair; p += blockDim.x) {
        const int m = t.pair_row[p], j = t.pair_col[p];
        const double4 y = t.pair_y[p];
        const double mr = s.vre[m], mi = s.vim[m], jr = s.vre[j], ji = s.vim[j];
        const double a = mr * jr + mi * ji, b = mi * jr - mr * ji;
        const bool mpq = t.node_pq[m], jpq = t.node_pq[j];
        const double ivm = mpq ? 1.0 / s.vmag[m] : 0.0, ivj = jpq ? 1.0 / s.vmag[j] : 0.0;
        const double u1 = y.x * b - y.y * a, u2 = y.x * a + y.y * b;        // block (m,j), Y_mj
        const double l1 = -y.z * b - y.w * a, l2 = y.z * a - y.w * b;       // block (j,m), Y_jm, theta_jm = -theta_mj
        Blk<T> U, L;
        U.a = T(u1);  U.b = T(u2 * ivj);  U.c = mpq ? T(-u2) : T(0);  U.d = mpq ? T(u1 * ivj) : T(0);
        L.a = T(l1);  L.b = T(l2 * ivm);  L.c = jpq ? T(-l2) : T(0);  L.d = jpq ? T(l1 * ivm) : T(0);
        st_blk(s.pr + 8 * p, U);
        st_blk(s.pr + 8 * p + 4, L);
    }
}

// a4 + forward half of a5: block LU on the static pattern, level by level (unit-lower L, pivot blocks D_m stored
// inverted), fused with the forward substitution L y = rhs which walks the same lists.  Contains barriers.
//   diag target m :  D_m = J(m,m) - sum_k L(m,k) U(k,m);   y_m = rhs_m - sum_k L(m,k) y_k      (k: pairs (k,m))
//   pair target p :  U(m,j) = J(m,j) - sum_k L(m,k) U(k,j);  L(j,m) = (J(j,m) - sum_k L(j,k) U(k,m)) D_m^-1
// transposed = true runs U^T w = g instead of L y = rhs:  w_m = D_m^-T (g_m - sum_k U(k,m)^T w_k).
template <typename T, bool kFactor, bool kSolve, bool kTransposed>
__device__ __forceinline__ void stage_factor_forward(const DevTemplate& t, const Scen<T>& s) {
    for (int l = 0; l < t.n_level; ++l) {
        const int m0 = t.level_ptr[l], m1 = t.level_ptr[l + 1];
        for (int m = m0 + threadIdx.x; m < m1; m += blockDim.x) {
            const int t0 = t.dterm_ptr[m], t1 = t.dterm_ptr[m + 1];
            Blk<T> D = ld_blk<T>(s.dg + 4 * m);
            T y0 = T(s.rhs[2 * m]), y1 = T(s.rhs[2 * m + 1]);
            for (int q = t0; q < t1; ++q) {
                const int a = t.dterm[q];
                const int k = t.pair_row[a];
                const Blk<T> U = ld_blk<T>(s.pr + 8 * a), L = ld_blk<T>(s.pr + 8 * a + 4);
                if (kFactor) mulsub(D, L, U);
                if (kSolve) {
                    const T x0 = T(s.rhs[2 * k]), x1 = T(s.rhs[2 * k + 1]);
                    if (!kTransposed) { y0 -= L.a * x0 + L.b * x1;  y1 -= L.c * x0 + L.d * x1; }
                    else              { y0 -= U.a * x0 + U.c * x1;  y1 -= U.b * x0 + U.d * x1; }
                }
            }
            if (kFactor) { D = inv(D); st_blk(s.dg + 4 * m, D); }
            if (kSolve) {
                if (kTransposed) { const T z0 = D.a * y0 + D.c * y1, z1 = D.b * y0 + D.d * y1; y0 = z0; y1 = z1; }
                s.rhs[2 * m] = double(y0);
                s.rhs[2 * m + 1] = double(y1);
            }
        }
        if (kFactor) {
            __syncthreads();
            const int p0 = t.pair_ptr[m0], p1 = t.pair_ptr[m1];
            for (int p = p0 + threadIdx.x; p < p1; p += blockDim.x) {
                Blk<T> U = ld_blk<T>(s.pr + 8 * p), L = ld_blk<T>(s.pr + 8 * p + 4);
                const int q1 = t.term_ptr[p + 1];
                for (int q = t.term_ptr[p]; q < q1; ++q) {
                    const int2 ab = t.term_ab[q];
                    mulsub(U, ld_blk<T>(s.pr + 8 * ab.x + 4), ld_blk<T>(s.pr + 8 * ab.y));
                    mulsub(L, ld_blk<T>(s.pr + 8 * ab.y + 4), ld_blk<T>(s.pr + 8 * ab.x));
                }
                L = mul(L, ld_blk<T>(s.dg + 4 * t.pair_row[p]));
                st_blk(s.pr + 8 * p, U);
                st_blk(s.pr + 8 * p + 4, L);
            }
        }
        __syncthreads();
    }
}

// backward half of a5: U x = y, i.e. x_m = D_m^-1 (y_m - sum_j U(m,j) x_j) over the pairs owned by m, levels
// descending.  transposed: L^T lambda = w, lambda_m = w_m - sum_j L(j,m)^T lambda_j.  Contains barriers.
template <typename T, bool kTransposed>
__device__ __forceinline__ void stage_backward(const DevTemplate& t, const Scen<T>& s) {
    for (int l = t.n_level - 1; l >= 0; --l) {
        const int m0 = t.level_ptr[l], m1 = t.level_ptr[l + 1];
        for (int m = m0 + threadIdx.x; m < m1; m += blockDim.x) {
            T y0 = T(s.rhs[2 * m]), y1 = T(s.rhs[2 * m + 1]);
            const int p1 = t.pair_ptr[m + 1];
            for (int p = t.pair_ptr[m]; p < p1; ++p) {
                const int j = t.pair_col[p];
                const T x0 = T(s.rhs[2 * j]), x1 = T(s.rhs[2 * j + 1]);
                if (!kTransposed) { const Blk<T> U = ld_blk<T>(s.pr + 8 * p); y0 -= U.a * x0 + U.b * x1; y1 -= U.c * x0 + U.d * x1; }
                else { const Blk<T> L = ld_blk<T>(s.pr + 8 * p + 4); y0 -= L.a * x0 + L.c * x1; y1 -= L.b * x0 + L.d * x1; }
            }
            if (!kTransposed) {
                const Blk<T> D = ld_blk<T>(s.dg + 4 * m);
                const T z0 = D.a * y0 + D.b * y1, z1 = D.c * y0 + D.d * y1; y0 = z0; y1 = z1;
            }
            s.rhs[2 * m] = double(y0);
            s.rhs[2 * m + 1] = double(y1);
        }
        __syncthreads();
    }
}

}  // namespace sable
