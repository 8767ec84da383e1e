// Staged (one kernel per stage, state in HBM/L2 between stages), adjoint and debug kernels.
#pragma once
#include "sable_kernels.cuh"

namespace sable {

// ---- staged mode: grid = batch, CTA b = scenario b, all arrays in the HBM workspace (placement 3 layout) -------
template <typename T>
__global__ void k_st_init(const SolveArgs A) {
    const int b = blockIdx.x;
    T* fac_b = reinterpret_cast<T*>(A.factors) + (size_t)b * A.fac_stride;
    const Scen<T> s = carve<T>(nullptr, 3, A.t.n_node, A.t.n_pair, A.work + (size_t)b * A.work_stride, fac_b);
    scen_init<T>(A, s, b);
    if (threadIdx.x == 0) { A.status[b] = 0; A.it[b] = 0; }
}

// a1 + a6 + a2: mismatch, norm, convergence decision, Jacobian fill for the scenarios that go on
template <typename T>
__global__ void k_st_mismatch_fill(const SolveArgs A) {
    __shared__ double red[32];
    const int b = blockIdx.x;
    if (A.status[b] != 0) return;                                   // masked: no loads, no stores
    T* fac_b = reinterpret_cast<T*>(A.factors) + (size_t)b * A.fac_stride;
    const Scen<T> s = carve<T>(nullptr, 3, A.t.n_node, A.t.n_pair, A.work + (size_t)b * A.work_stride, fac_b);
    const double r = cta_max_nan(stage_mismatch<T>(A.t, s, true), red);
    const int it = A.it[b];
    int st = 0;
    if (r <= A.tol) st = 1;
    else if (it == A.max_it || !(fabs(r) < __longlong_as_double(0x7ff0000000000000LL))) st = 2;
    if (st == 0 || A.keep) stage_fill_pairs<T>(A.t, s);
    if (st != 0) {
        __syncthreads();
        if (threadIdx.x == 0) {
            A.status[b] = st;
            A.iterations[b] = st == 1 ? it : A.max_it;
            A.converged[b] = st == 1;
            if (A.final_norm) A.final_norm[b] = r;
        }
        const size_t o = (size_t)b * A.t.n_bus;
        for (int m = threadIdx.x; m <= A.t.n_node; m += blockDim.x) {
            const int bus = A.t.node_bus[m];
            A.vm[o + bus] = s.vmag[m]; A.va[o + bus] = s.ang[m];
        }
        if (A.keep) { __syncthreads(); stage_factor_forward<T, true, false, false>(A.t, s); }
    }
}

// a4 + a5: refactor, forward/backward substitution, FP64 state update
template <typename T>
__global__ void k_st_factor_solve(const SolveArgs A) {
    const int b = blockIdx.x;
    if (A.status[b] != 0) return;
    T* fac_b = reinterpret_cast<T*>(A.factors) + (size_t)b * A.fac_stride;
    const Scen<T> s = carve<T>(nullptr, 3, A.t.n_node, A.t.n_pair, A.work + (size_t)b * A.work_stride, fac_b);
    stage_factor_forward<T, true, true, false>(A.t, s);
    stage_backward<T, false>(A.t, s);
    scen_update<T>(A.t, s);
    if (threadIdx.x == 0) A.it[b] += 1;
}

// ---- adjoint / generic linear solve on stored factors ---------------------------------------------------------
struct LinArgs {
    DevTemplate t;
    int32_t batch, transposed;
    const double *rhs_p, *rhs_q;      // [batch][n_bus]: theta/P component and Vm/Q component per bus
    double *x_p, *x_q;
    const void* factors; int64_t fac_stride;
};

// a7: J1^T lambda = g with the kept factors (eq. 14): U^T w = g ascending, L^T lambda = w descending.
// rhs lives in shared memory when it fits (use_smem), else in the caller's x_p/x_q is not usable -> work buffer.
template <typename T>
__global__ void k_linsolve(const LinArgs A, double* work, int64_t work_stride, int use_smem) {
    extern __shared__ __align__(16) unsigned char smem[];
    const DevTemplate& t = A.t;
    const int b = blockIdx.x;
    Scen<T> s{};
    s.rhs = use_smem ? reinterpret_cast<double*>(smem) : work + (size_t)b * work_stride;
    T* f = const_cast<T*>(reinterpret_cast<const T*>(A.factors)) + (size_t)b * A.fac_stride;
    s.dg = f; s.pr = f + 4 * t.n_node;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x; m < t.n_node; m += blockDim.x) {
        const int bus = t.node_bus[m];
        s.rhs[2 * m] = A.rhs_p[o + bus];
        s.rhs[2 * m + 1] = t.node_pq[m] ? A.rhs_q[o + bus] : 0.0;
    }
    __syncthreads();
    if (A.transposed) { stage_factor_forward<T, false, true, true>(t, s); stage_backward<T, true>(t, s); }
    else              { stage_factor_forward<T, false, true, false>(t, s); stage_backward<T, false>(t, s); }
    for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
        const int bus = t.node_bus[m];
        A.x_p[o + bus] = m < t.n_node ? s.rhs[2 * m] : 0.0;
        A.x_q[o + bus] = (m < t.n_node && t.node_pq[m]) ? s.rhs[2 * m + 1] : 0.0;
    }
}

// ---- debug: state from caller's (vm, va), mismatch / Jacobian / refactor at that state ---------------------------
struct DebugArgs {
    DevTemplate t;
    int32_t batch, what;              // what: 0 mismatch, 1 jacobian, 2 refactor only (factors kept for k_linsolve)
    const double *p_spec, *q_spec, *vm, *va;
    double *f_p, *f_q, *norm, *diag, *pairs;
    void* factors; double* work; int64_t fac_stride, work_stride;
};

template <typename T>
__global__ void k_debug(const DebugArgs A) {
    __shared__ double red[32];
    const DevTemplate& t = A.t;
    const int b = blockIdx.x;
    T* fac_b = reinterpret_cast<T*>(A.factors) + (size_t)b * A.fac_stride;
    const Scen<T> s = carve<T>(nullptr, 3, t.n_node, t.n_pair, A.work + (size_t)b * A.work_stride, fac_b);
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
        const int bus = t.node_bus[m];
        const double vm = A.vm[o + bus], th = A.va[o + bus];
        double sn, cs; sincos(th, &sn, &cs);
        s.vmag[m] = vm; s.ang[m] = th; s.vre[m] = vm * cs; s.vim[m] = vm * sn;
        if (m < t.n_node) { s.psp[m] = A.p_spec ? A.p_spec[o + bus] : 0.0; s.qsp[m] = A.q_spec ? A.q_spec[o + bus] : 0.0; }
    }
    __syncthreads();
    const double r = cta_max_nan(stage_mismatch<T>(t, s, true), red);
    if (A.what == 0) {
        for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
            const int bus = t.node_bus[m];
            A.f_p[o + bus] = m < t.n_node ? -s.rhs[2 * m] : 0.0;
            A.f_q[o + bus] = m < t.n_node ? -s.rhs[2 * m + 1] : 0.0;
        }
        if (threadIdx.x == 0) A.norm[b] = r;
        return;
    }
    stage_fill_pairs<T>(t, s);
    __syncthreads();
    if (A.what == 1) {
        for (int i = threadIdx.x; i < 4 * t.n_node; i += blockDim.x) A.diag[(size_t)b * 4 * t.n_node + i] = double(s.dg[i]);
        for (int i = threadIdx.x; i < 8 * t.n_pair; i += blockDim.x) A.pairs[(size_t)b * 8 * t.n_pair + i] = double(s.pr[i]);
        return;
    }
    stage_factor_forward<T, true, false, false>(t, s);
}

}  // namespace sable
