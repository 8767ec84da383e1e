// Kernels of the batched NR power flow: the fused persistent kernel (whole NR loop of a scenario on one CTA,
// scenarios pulled from an atomic queue = convergence masking by construction), the staged per-stage kernels
// (profiling mode), the adjoint kernel and the debug kernels.  Launched from sable_capi.cu.
#pragma once
#include "sable_stages.cuh"

namespace sable {

struct SolveArgs {
    DevTemplate t;
    int32_t batch, max_it, keep, placement;
    double tol;
    const double *p_spec, *q_spec, *v_set, *vm0, *va0;     // [batch][n_bus]
    double *vm, *va, *final_norm;
    int32_t* iterations;
    uint8_t* converged;
    void* factors;            // [max_batch][fac_stride] of T
    double* work;             // [max_batch][work_stride]
    int64_t fac_stride, work_stride;
    int32_t* queue;           // persistent-kernel scenario counter
    int32_t* status;          // staged mode: [batch] 0 = active, 1 = converged, 2 = stopped
    int32_t* it;              // staged mode: [batch]
};

__host__ __device__ inline int state_len(int n_node) { return (n_node + 2) & ~1; }          // padded array length
__host__ __device__ inline int64_t work_doubles(int n_node) { return 8 * (int64_t)state_len(n_node); }
__host__ __device__ inline int64_t fac_elems(int n_node, int n_pair) { return 4 * (int64_t)n_node + 8 * (int64_t)n_pair; }
// dynamic shared memory (bytes) a placement needs, incl. 32 doubles of reduction scratch
template <typename T> __host__ __device__ inline int64_t smem_need(int placement, int n_node, int n_pair) {
    const int64_t na = state_len(n_node);
    int64_t b = 32 * 8;
    if (placement <= 1) b += 8 * na * 8;
    else if (placement == 2) b += 2 * na * 8;              // rhs only
    if (placement == 0) b += fac_elems(n_node, n_pair) * (int64_t)sizeof(T);
    return b;
}

// placement 0: all in smem; 1: factors in HBM, state + rhs in smem; 2: rhs in smem, rest in HBM/L2; 3: all in HBM/L2
template <typename T>
__device__ __forceinline__ Scen<T> carve(unsigned char* smem, int placement, int n_node, int n_pair, double* work_b, T* fac_b) {
    const int na = state_len(n_node);
    double* sm = reinterpret_cast<double*>(smem) + 32;
    Scen<T> s;
    double* st = (placement <= 1) ? sm : work_b;
    s.vre = st; s.vim = st + na; s.vmag = st + 2 * na; s.ang = st + 3 * na; s.psp = st + 4 * na; s.qsp = st + 5 * na;
    s.rhs = (placement <= 1) ? sm + 6 * na : (placement == 2 ? sm : work_b + 6 * na);
    T* f = (placement == 0) ? reinterpret_cast<T*>(sm + 8 * na) : fac_b;
    s.dg = f; s.pr = f + 4 * n_node;
    return s;
}

template <typename T>
__device__ __forceinline__ void scen_init(const SolveArgs& A, const Scen<T>& s, int b) {
    const DevTemplate& t = A.t;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {       // PAPER.md:287 flat start unless vm0/va0 given
        const int bus = t.node_bus[m];
        const bool pq = m < t.n_node && t.node_pq[m];
        const double vm = pq ? (A.vm0 ? A.vm0[o + bus] : 1.0) : A.v_set[o + bus];
        const double th = A.va0 ? A.va0[o + bus] : 0.0;
        double sn, cs; sincos(th, &sn, &cs);
        s.vmag[m] = vm; s.ang[m] = th; s.vre[m] = vm * cs; s.vim[m] = vm * sn;
        if (m < t.n_node) { s.psp[m] = A.p_spec[o + bus]; s.qsp[m] = pq ? A.q_spec[o + bus] : 0.0; }
    }
}

template <typename T>
__device__ __forceinline__ void scen_update(const DevTemplate& t, const Scen<T>& s) {   // PAPER.md:90, FP64 accumulate
    for (int m = threadIdx.x; m < t.n_node; m += blockDim.x) {
        const double th = s.ang[m] + s.rhs[2 * m];
        const double vm = t.node_pq[m] ? s.vmag[m] + s.rhs[2 * m + 1] : s.vmag[m];
        double sn, cs; sincos(th, &sn, &cs);
        s.ang[m] = th; s.vmag[m] = vm; s.vre[m] = vm * cs; s.vim[m] = vm * sn;
    }
}

template <typename T>
__device__ __forceinline__ void scen_finish(const SolveArgs& A, const Scen<T>& s, int b, int it, bool conv, double r,
                                            T* fac_b) {
    const DevTemplate& t = A.t;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
        const int bus = t.node_bus[m];
        A.vm[o + bus] = s.vmag[m]; A.va[o + bus] = s.ang[m];
    }
    if (threadIdx.x == 0) {
        A.iterations[b] = conv ? it : A.max_it;
        A.converged[b] = conv ? 1 : 0;
        if (A.final_norm) A.final_norm[b] = r;
    }
    if (A.keep) {        // factors of J1 at the final iterate for the adjoint (reading 16)
        stage_fill_pairs<T>(t, s);
        __syncthreads();
        stage_factor_forward<T, true, false, false>(t, s);
        if (s.dg != fac_b) {
            const int64_t n4 = fac_elems(t.n_node, t.n_pair) / 4;
            for (int64_t i = threadIdx.x; i < n4; i += blockDim.x) st_blk(fac_b + 4 * i, ld_blk<T>(s.dg + 4 * i));
        }
    }
}

// Fused persistent kernel: loop of DESIGN.md "NR loop convention", all state on chip / in L2.
template <typename T>
__global__ void __launch_bounds__(1024) k_nr_fused(const SolveArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ int s_b;
    double* red = reinterpret_cast<double*>(smem);
    const DevTemplate& t = A.t;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_b = atomicAdd(A.queue, 1);
        __syncthreads();
        const int b = s_b;
        if (b >= A.batch) return;
        T* fac_b = reinterpret_cast<T*>(A.factors) + (size_t)b * A.fac_stride;
        const Scen<T> s = carve<T>(smem, A.placement, t.n_node, t.n_pair, A.work + (size_t)b * A.work_stride, fac_b);
        scen_init<T>(A, s, b);
        __syncthreads();
        int it = 0; bool conv = false; double r;
        for (;;) {
            r = cta_max_nan(stage_mismatch<T>(t, s, true), red);
            if (r <= A.tol) { conv = true; break; }
            if (it == A.max_it || !(fabs(r) < __longlong_as_double(0x7ff0000000000000LL))) break;
            stage_fill_pairs<T>(t, s);
            __syncthreads();
            stage_factor_forward<T, true, true, false>(t, s);
            stage_backward<T, false>(t, s);
            scen_update<T>(t, s);
            __syncthreads();
            ++it;
        }
        scen_finish<T>(A, s, b, it, conv, r, fac_b);
    }
}

}  // namespace sable
