// Device-side view of the shared fixed-pattern template and the per-scenario stage routines of the batched
// Newton-Raphson power flow (eq. 6-8, eq. 14).  One CTA works on one scenario; every routine below is
// a CTA-wide cooperative step that ends WITHOUT a barrier unless stated.  The same routines serve the fused
// persistent kernel and the staged per-stage kernels (sable_kernels.cu).
//
// Block conventions.  Every non-slack bus is a node with a 2x2 block: rows (P_m, Q_m), columns (theta_m, Vm_m),
// stored row-major [dP/dth, dP/dVm, dQ/dth, dQ/dVm].  A PV node keeps the block with the Q row and Vm column
// padded (0 off the diagonal, 1 on it).  Per scenario the factor storage is
//   dg[4*n_node]   : J(m,m), then after refactor the INVERSE of the pivot block D_m
//   pr[8*n_pair]   : pair p = (m,j), m < j:  pr[8p..8p+3] = J(m,j) -> U(m,j);  pr[8p+4..8p+7] = J(j,m) -> L(j,m)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace sable {

struct DevTemplate {
    int32_t n_bus, n_node, n_pair, n_level, slack;
    const int32_t* level_ptr;   // [n_level+1]
    const int32_t* node_bus;    // [n_node+1]  (entry n_node = slack bus)
    const uint8_t* node_pq;     // [n_node]
    const int32_t* yptr;        // [n_node+1]  Y rows of the non-slack buses in node order
    const int32_t* ycol;        // node positions (slack = n_node)
    const double2* ygb;         // (G, B) per stored Y entry
    const double2* ydiag_gb;    // [n_node] (G_mm, B_mm)
    const int32_t* pair_ptr;    // [n_node+1]
    const int32_t* pair_row;    // [n_pair]
    const int32_t* pair_col;    // [n_pair]
    const double4* pair_y;      // [n_pair] (G_mj, B_mj, G_jm, B_jm); zeros for a fill pair
    const int32_t* term_ptr;    // [n_pair+1]
    const int2*    term_ab;     // [n_term] (pair (k,m), pair (k,j))
    const int32_t* dterm_ptr;   // [n_node+1]
    const int32_t* dterm;       // [n_pair]
};

template <typename T> struct Blk { T a, b, c, d; };   // [[a b][c d]]

template <typename T> __device__ __forceinline__ Blk<T> ld_blk(const T* p);
template <> __device__ __forceinline__ Blk<double> ld_blk<double>(const double* p) {
    double2 x = *reinterpret_cast<const double2*>(p), y = *reinterpret_cast<const double2*>(p + 2);
    return {x.x, x.y, y.x, y.y};
}
template <> __device__ __forceinline__ Blk<float> ld_blk<float>(const float* p) {
    float4 x = *reinterpret_cast<const float4*>(p);
    return {x.x, x.y, x.z, x.w};
}
__device__ __forceinline__ void st_blk(double* p, const Blk<double>& v) {
    *reinterpret_cast<double2*>(p) = make_double2(v.a, v.b);
    *reinterpret_cast<double2*>(p + 2) = make_double2(v.c, v.d);
}
__device__ __forceinline__ void st_blk(float* p, const Blk<float>& v) {
    *reinterpret_cast<float4*>(p) = make_float4(v.a, v.b, v.c, v.d);
}
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

// CTA-wide max of a non-negative value; NaN-propagating (a NaN anywhere gives NaN, like the paper's ||F||inf on a
// diverged iterate, reading 18).  `red` is a shared array of >= 32 doubles.  Contains barriers.
__device__ __forceinline__ double cta_max_nan(double v, double* red) {
    auto mx = [](double x, double y) { return (x != x || y != y) ? __longlong_as_double(0x7ff8000000000000LL) : fmax(x, y); };
    for (int o = 16; o > 0; o >>= 1) v = mx(v, __shfl_xor_sync(0xffffffffu, v, o));
    int w = threadIdx.x >> 5, l = threadIdx.x & 31, nw = (blockDim.x + 31) >> 5;
    __syncthreads();
    if (l == 0) red[w] = v;
    __syncthreads();
    v = l < nw ? red[l] : 0.0;
    for (int o = 16; o > 0; o >>= 1) v = mx(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

}  // namespace sable
