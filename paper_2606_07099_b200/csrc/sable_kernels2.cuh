// Staged kernels (one kernel per stage, state in HBM between stages -- the per-stage profiling mode), the adjoint /
// linear-solve kernel on kept factors, and the debug kernels.  The staged kernels run the fused kernel's own stage
// routines in the fused kernel's workspace layout (one CTA per group of G scenarios, slots in lockstep); the debug
// kernels serve one scenario per CTA (gsh = 0).
#pragma once
#include "sable_kernels.cuh"

namespace sable {

// everything in the HBM slices of scenario b's group
template <typename T>
__device__ __forceinline__ Slot<T, 2> hbm_slot(const DevTemplate& t, char* factors, int64_t fac_stride, char* work, int64_t work_stride, int b, int gsh = 0) {
    Slot<T, 2> s = carve<T, 2>(nullptr, 0, t.n_node, t.n_pair, gsh, 0);
    s.sb = nullptr;
    bind<T, 2>(s, factors, fac_stride, work, work_stride, b);
    return s;
}

// index program read in place (no shared-memory ring)
__device__ __forceinline__ BlobRing no_ring(const DevTemplate& t) {
    BlobRing r;
    r.slots = nullptr; r.mbar = nullptr; r.gblob = t.blob; r.lv = t.level; r.R = 0; r.slot_bytes = 0;
    r.first = t.n_level; r.n_level = t.n_level; r.use = 0; r.tim = nullptr; r.on = false;
    return r;
}

constexpr int kStageScratch = 32 * 8 * kBigDoubles;   // doubles: big-target partials of up to 32 warps x 8 slots

template <typename T>
__global__ void k_st_init(const SolveArgs A) {
    const int gsh = A.gsh, g = threadIdx.x & ((1 << gsh) - 1), b = (blockIdx.x << gsh) + g;
    if (b >= A.batch) return;
    const Slot<T, 2> s = hbm_slot<T>(A.t, A.factors, A.fac_stride, A.work, A.work_stride, b, gsh);
    scen_init<T, 2>(A, s, b, threadIdx.x >> gsh, blockDim.x >> gsh);
    if ((threadIdx.x >> gsh) == 0) { A.status[b] = 0; A.it[b] = 0; }
}

// a1 + a6 + a2: mismatch, norm, convergence decision, Jacobian fill (in place, into the factor value array) for the
// scenarios that go on; a scenario that finishes with keep_factors gets its factors of J1 at the final iterate here.
// Masked slots (finished earlier, or beyond the batch) run along on the spare workspace group.
// (kThreads, kCtas: the register budget -- up to 128 threads x 7 CTAs per SM (72 registers), as the fused kernel's small
// variant, or up to 512 x 2 (64))
template <typename T, int kThreads, int kCtas>
__global__ void __launch_bounds__(kThreads, kCtas) k_st_mismatch_fill(const SolveArgs A) {
    __shared__ double red[32 * 32];
    __shared__ double scratch[kStageScratch];
    const DevTemplate& t = A.t;
    const int gsh = A.gsh, G = 1 << gsh, g = threadIdx.x & (G - 1), tsub = threadIdx.x >> gsh, nsub = blockDim.x >> gsh;
    const int bb = (blockIdx.x << gsh) + g;
    const bool act = bb < A.batch && A.status[bb] == 0;
    if (!__syncthreads_or(act)) return;                              // whole group masked: no loads, no stores
    const int trash = (A.trash_grp << gsh) + g;
    Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, act ? bb : trash, gsh);
    PivotFlag pf{act ? A.pivot + bb : nullptr};
    if (act && tsub == 0) atomicAnd(pf.w, 1);
    __syncthreads();
    const size_t row = (size_t)(act ? bb : 0) * t.n_bus;
    const double r = slot_max_nan(stage_mismatch<T, 2>(t, s, A.p_spec + row, A.q_spec + row, act, t.level[0].m1, pf, Team{0, 1}), red, gsh);
    int st = 0;
    if (act) {
        const int it = A.it[bb];
        if (r <= A.tol) st = 1;
        else if (it == A.max_it || !(fabs(r) < __longlong_as_double(0x7ff0000000000000LL))) st = 2;
        if (st != 0) {
            scen_output<T, 2>(A, s, bb, it, st == 1, r, tsub, nsub);
            if (tsub == 0) A.status[bb] = st;
        } else if (tsub == 0) atomicAdd(A.active + A.stage_it, 1);
    }
    const bool go_on = act && st == 0, fin = act && st != 0 && A.keep;
    if (!go_on && !fin) { bind<T, 2>(s, A.factors, A.fac_stride, A.work, A.work_stride, trash); pf.w = nullptr; }
    __syncthreads();                                                 // scen_output has read the state the fill's trash lanes may overwrite
    stage_fill_pairs<T, 2>(t, s, tsub, nsub);
    if (!__syncthreads_or(fin)) return;                              // (the barrier also orders the J stores before the refactor)
    if (!fin) { bind<T, 2>(s, A.factors, A.fac_stride, A.work, A.work_stride, trash); pf.w = nullptr; }
    BlobRing ring = no_ring(t);
    stage_factor_forward<T, 2, true, false, false, true>(t, s, t.level, ring, pf, scratch, Team{0, 1});
}

// a4 + a5: refactor, forward/backward substitution, FP64 state update
template <typename T, int kThreads, int kCtas>
__global__ void __launch_bounds__(kThreads, kCtas) k_st_factor_solve(const SolveArgs A) {
    __shared__ double scratch[kStageScratch];
    const DevTemplate& t = A.t;
    const int gsh = A.gsh, G = 1 << gsh, g = threadIdx.x & (G - 1), tsub = threadIdx.x >> gsh, nsub = blockDim.x >> gsh;
    const int bb = (blockIdx.x << gsh) + g;
    const bool act = bb < A.batch && A.status[bb] == 0;
    if (!__syncthreads_or(act)) return;
    const Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, act ? bb : (A.trash_grp << gsh) + g, gsh);
    const PivotFlag pf{act ? A.pivot + bb : nullptr};
    BlobRing ring = no_ring(t);
    stage_factor_forward<T, 2, true, true, false, true>(t, s, t.level, ring, pf, scratch, Team{0, 1});
    stage_backward<T, 2, false>(t, s, t.level, ring, Team{0, 1});
    if (A.ir) return;                                                // the step stays in rh: refined, then applied by k_st_ir_update
    stage_update<T, 2>(t, s, tsub, nsub);
    if (act && tsub == 0) A.it[bb] += 1;
}

// ---- inner iterative refinement of the forward linear solve (sable_options.ir_sweeps; SURVEY.md section 8(c) reading 15:
// r = -F1 - J1 dz with J1 and F1 in FP64, correction solved on the FP32 factors, added in FP64; PAPER.md:255-271 is the
// mixed-precision scheme this refines -- the paper itself has no inner sweeps).  Three small kernels around k_linsolve:
// export of the state and the FP32-solved step to bus-order arrays, the FP64 residual evaluated from Y_bus and V with the
// Alg. 1 formulas (no stored FP64 Jacobian), and the update z1 += dz (eq. 8).
// (tiles of 1024 / G buses go through shared memory: the slots interleave the G scenarios of a group node by node, the
// bus-order arrays are scenario-major -- reads are coalesced over the scenarios of a node, writes over the buses of a scenario)
constexpr int kIrTile = 1024;
template <typename T>
__global__ void k_st_ir_export(const SolveArgs A) {
    __shared__ double2 tv[kIrTile + kIrTile / 8];
    __shared__ double tvm[kIrTile + kIrTile / 8], tdp[kIrTile + kIrTile / 8], tdq[kIrTile + kIrTile / 8];
    const DevTemplate& t = A.t;
    const int gsh = A.gsh, G = 1 << gsh, g = threadIdx.x & (G - 1), b = (blockIdx.x << gsh) + g;
    const bool act = b < A.batch && A.status[b] == 0;
    if (!__syncthreads_or(act)) return;
    const Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, act ? b : (blockIdx.x << gsh), gsh);
    const int tb = kIrTile >> gsh;                                   // buses per tile; entry (bus bi, slot g) at bi * G + g (+ padding)
    for (int i0 = 0; i0 < t.n_bus; i0 += tb) {
        for (int idx = threadIdx.x; idx < kIrTile; idx += blockDim.x) {      // blockDim is a multiple of G: idx & (G - 1) == g
            const int i = i0 + (idx >> gsh);
            if (act && i < t.n_bus) {
                const int m = A.ir_bus_node[i], e = idx + (idx >> 3);
                const double2 dz = m < t.n_node ? s.rh(m) : make_double2(0.0, 0.0);
                tv[e] = s.vv(m);
                tvm[e] = s.ma(m).x;
                tdp[e] = dz.x;
                tdq[e] = (m < t.n_node && t.node_pq[m]) ? dz.y : 0.0;
            }
        }
        __syncthreads();
        for (int idx = threadIdx.x; idx < kIrTile; idx += blockDim.x) {      // bus fastest
            const int bi = idx & (tb - 1), gg = idx >> (10 - gsh), i = i0 + bi, bb = (blockIdx.x << gsh) + gg;
            if (i < t.n_bus && bb < A.batch && A.status[bb] == 0) {
                const int q = (bi << gsh) + gg, e = q + (q >> 3);
                const size_t o = (size_t)bb * t.n_bus + i;
                A.ir_v[o] = tv[e]; A.ir_vm[o] = tvm[e]; A.ir_dzp[o] = tdp[e]; A.ir_dzq[o] = tdq[e];
            }
        }
        __syncthreads();
    }
}

template <typename T>
__global__ void k_st_ir_update(const SolveArgs A) {
    const int gsh = A.gsh, g = threadIdx.x & ((1 << gsh) - 1), b = (blockIdx.x << gsh) + g;
    if (b >= A.batch || A.status[b] != 0) return;
    const DevTemplate& t = A.t;
    const Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, b, gsh);
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x >> gsh; m < t.n_node; m += blockDim.x >> gsh) {
        const int bus = t.node_bus[m];
        const double2 a = s.ma(m);
        const double th = a.y + A.ir_dzp[o + bus], vm = t.node_pq[m] ? a.x + A.ir_dzq[o + bus] : a.x;
        double sn, cs; sincos(th, &sn, &cs);
        s.set_ma(m, make_double2(vm, th));
        s.set_vv(m, make_double2(vm * cs, vm * sn));
    }
    if ((threadIdx.x >> gsh) == 0) A.it[b] += 1;
}

struct IrArgs {
    int32_t n_bus, batch;
    const int32_t *fptr, *fcol;       // full Y_bus CSR, bus order
    const double2* fgb;
    const uint8_t* bus_type;          // 0 PQ, 1 PV, 2 slack
    const int32_t* status;            // [batch] 0 = scenario still iterating
    const double *p_spec, *q_spec;    // [batch][n_bus]
    const double2* v;
    const double *vm, *dzp, *dzq;
    double *rp, *rq;                  // out: r = -F1 - J1 dz, rows P (non-slack) and Q (PQ); zero elsewhere and for finished scenarios
    const int32_t* long_rows; int32_t n_long;   // buses whose Y_bus row has more than kLongRowIr entries
};

// one row of Y_bus per thread (a whole warp for rows above kLongRowIr entries): the row sum gives the calculated injection
// (F1 row, eq. 6) and, entry by entry, the off-diagonal blocks of J1 applied to the neighbour's step; the diagonal block uses
// the calculated P_i, Q_i
constexpr int kLongRowIr = 32;
__device__ __forceinline__ double warp_sum_ir(double x) {
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
__device__ __forceinline__ void ir_row(const IrArgs& A, int b, int i, bool warp) {
    const size_t o = (size_t)b * A.n_bus;
    const int ti = A.bus_type[i], lane = threadIdx.x & 31;
    double rp = 0.0, rq = 0.0;
    if (ti != 2 && A.status[b] == 0) {
        const double2 vi = A.v[o + i];
        double ire = 0.0, iim = 0.0, ap = 0.0, aq = 0.0, ydx = 0.0, ydy = 0.0;
        for (int k = A.fptr[i] + (warp ? lane : 0); k < A.fptr[i + 1]; k += warp ? 32 : 1) {
            const int j = A.fcol[k];
            const double2 y = A.fgb[k], x = A.v[o + j];
            const double tr = y.x * x.x - y.y * x.y, tim = y.y * x.x + y.x * x.y;
            ire += tr; iim += tim;
            if (j == i) { ydx = y.x; ydy = y.y; continue; }
            const double u2 = vi.x * tr + vi.y * tim, u1 = vi.y * tr - vi.x * tim;
            const double dth = A.dzp[o + j], dvm = A.dzq[o + j] / A.vm[o + j];            // zero where the column is not in z1
            ap += u1 * dth + u2 * dvm;
            aq += -u2 * dth + u1 * dvm;
        }
        if (warp) { ire = warp_sum_ir(ire); iim = warp_sum_ir(iim); ap = warp_sum_ir(ap); aq = warp_sum_ir(aq); ydx = warp_sum_ir(ydx); ydy = warp_sum_ir(ydy); }
        const double P = vi.x * ire + vi.y * iim, Q = vi.y * ire - vi.x * iim;
        const double vm = A.vm[o + i], v2 = vm * vm, dth = A.dzp[o + i], dvm = A.dzq[o + i];
        ap += (-Q - ydy * v2) * dth + (P / vm + ydx * vm) * dvm;
        aq += (P - ydx * v2) * dth + (Q / vm - ydy * vm) * dvm;
        rp = (A.p_spec[o + i] - P) - ap;
        if (ti == 0) rq = (A.q_spec[o + i] - Q) - aq;
    }
    if (warp && lane) return;
    A.rp[o + i] = rp; A.rq[o + i] = rq;
}
__global__ void k_ir_residual(const IrArgs A) {
    const size_t total = (size_t)A.batch * A.n_bus;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int b = (int)(idx / A.n_bus), i = (int)(idx - (size_t)b * A.n_bus);
        if (A.fptr[i + 1] - A.fptr[i] <= kLongRowIr) ir_row(A, b, i, false);
    }
    const size_t nw = ((size_t)gridDim.x * blockDim.x) >> 5, tot = (size_t)A.batch * A.n_long;
    for (size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < tot; w += nw)
        ir_row(A, (int)(w / A.n_long), A.long_rows[w % A.n_long], true);
}

// ---- adjoint / generic linear solve on stored factors ---------------------------------------------------------
struct LinArgs {
    DevTemplate t;
    int32_t batch, transposed, rhs_in_smem, gsh;   // gsh: group size (log2) of the factor layout = that of the kernel that wrote them
    const double *rhs_p, *rhs_q;      // [batch][n_bus]: theta/P component and Vm/Q component per bus
    double *x_p, *x_q;
    const int32_t* pivot;             // tiny-pivot flags of the kept factors (bit 1), or nullptr
    char* factors; char* work; int64_t fac_stride, work_stride;
    int32_t big_off;                  // big-target scratch at the start of dynamic shared memory, right-hand sides behind it
    int32_t csz;                      // CTAs per team (cluster size); the right-hand sides then live in the group's workspace slice
    int32_t front_k, front_f0, front_level;   // dense top front of the transposed sweeps (0 = none): the last levels in shared memory
    int64_t front_off;
    LevelDesc front;
};

// a7: J1^T lambda = g with the kept factors (eq. 14): U^T w = g ascending, (L' D^-1)^T lambda = w descending.
// One CTA per group of G scenarios in lockstep (lane layout as in the NR kernel): factors stream from the group's
// interleaved HBM slices (coalesced; U only in the first sweep, L' only in the second), the right-hand sides live in
// shared memory when they fit.  A scenario whose kept factors carry a tiny-pivot flag gets NaN (its lambda would be
// garbage that nothing else reveals: the adjoint has no residual test).
template <typename T>
__global__ void __launch_bounds__(1024, 1) k_linsolve(const LinArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const DevTemplate& t = A.t;
    const Team tm{A.csz > 1 ? cluster_ctarank() : 0, A.csz > 1 ? A.csz : 1};
    const int gsh = A.gsh, G = 1 << gsh, g = threadIdx.x & (G - 1);
    const int nsub = (blockDim.x >> gsh) * tm.csz, tsub = tm.rank * (blockDim.x >> gsh) + (threadIdx.x >> gsh);
    const int bb = ((blockIdx.x / tm.csz) << gsh) + g;
    const bool act = bb < A.batch;
    Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, bb, gsh);
    double* scratch = reinterpret_cast<double*>(smem);
    if (A.rhs_in_smem) { s.gw = reinterpret_cast<char*>(smem) + A.big_off + g * 16; s.go_rh = 0; }   // only rh is touched: generic loads from shared memory
    const size_t o = (size_t)(act ? bb : 0) * t.n_bus;
    for (int m = tsub; m < t.n_node; m += nsub) {
        const int bus = t.node_bus[m];
        s.set_rh(m, act ? make_double2(A.rhs_p[o + bus], t.node_pq[m] ? A.rhs_q[o + bus] : 0.0) : make_double2(0.0, 0.0));
    }
    team_sync(tm);
    BlobRing ring = no_ring(t);
    const PivotFlag pf{nullptr};
    if (A.transposed && A.front_k > 0) {
        // the last elimination levels as one dense block matrix in shared memory (sable_front.cuh): two short loops of
        // shared-memory steps instead of two barrier-separated, memory-latency-bound phases per level
        const int tsub_c = threadIdx.x >> gsh, nsub_c = blockDim.x >> gsh;
        const Front<T> F = carve_front<T>(smem, A.front_off, A.front_k, A.front_f0, gsh, g);
        front_zero<T>(F, tsub_c, nsub_c);
        stage_factor_forward<T, 2, false, true, true, false, false>(t, s, t.level, ring, pf, scratch, tm, A.front_level);
        front_load<T, 2>(t, s, F, A.front, tsub_c, nsub_c);
        const FrontSink<T> sink{F, pf};
        accumulate_level<T, 2, false, true, true>(s, A.front, t.blob + A.front.blob_off, sink, pf, scratch, tm);
        __syncthreads();
        front_forward_t<T>(F, tsub_c, nsub_c);
        front_backward_t<T, 2>(s, F, tsub_c, nsub_c);
        stage_backward<T, 2, true, false>(t, s, t.level, ring, tm, A.front_level);
    }
    else if (A.transposed) { stage_factor_forward<T, 2, false, true, true, false>(t, s, t.level, ring, pf, scratch, tm); stage_backward<T, 2, true>(t, s, t.level, ring, tm); }
    else              { stage_factor_forward<T, 2, false, true, false, false>(t, s, t.level, ring, pf, scratch, tm); stage_backward<T, 2, false>(t, s, t.level, ring, tm); }
    if (act) {
        const bool bad = A.pivot && (A.pivot[bb] & 2);
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        for (int m = tsub; m <= t.n_node; m += nsub) {
            const int bus = t.node_bus[m];
            const double2 x = m < t.n_node ? s.rh(m) : make_double2(0.0, 0.0);
            A.x_p[o + bus] = m < t.n_node ? (bad ? nan : x.x) : 0.0;
            A.x_q[o + bus] = (m < t.n_node && t.node_pq[m]) ? (bad ? nan : x.y) : 0.0;
        }
    }
    if (tm.csz > 1) team_sync(tm);
}

// ---- Step-2 explicit recovery (PAPER.md:80 eq. 5, :95-99 eq. 9): with dF2/dz2 = I the block z2 = [p_g at the slack;
// q_g at PV and slack buses] is read off the calculated injections S = V o conj(Y_bus V) at the solved voltages.
// The kernel returns P_i(V), Q_i(V) for EVERY bus (net injection = generation - load); the caller picks
// the slack / PV rows.  One CTA per scenario: V in rectangular form goes to shared memory (or to the scenario's
// workspace slice when the grid is too large), then one row of Y_bus per thread.
struct RecoverArgs {
    int32_t n_bus, batch, v_in_smem;
    const int32_t *fptr, *fcol;
    const double2* fgb;                // (G, B) per stored entry, bus order
    const double *vm, *va;             // [batch][n_bus]
    double *p_inj, *q_inj;             // [batch][n_bus]
    char* work; int64_t work_stride;   // used when V does not fit shared memory
    const int32_t* long_rows; int32_t n_long;   // buses whose Y_bus row has more than kLongRow entries (served by a whole warp)
};

// A row of Y_bus with hundreds of entries (a hub bus) walked by one thread is a chain of dependent gathers that alone takes
// longer than everything else in these kernels (config 5: longest row 322 entries, ~0.1 ms): rows above kLongRow entries are
// left out of the thread-per-row passes and served by a whole warp each (lanes take every 32nd entry, shuffle reduction).
constexpr int kLongRow = 32;
__device__ __forceinline__ double warp_sum(double x) {
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}
// I_i = sum_k Y_ik V_k over the entries k0, k0 + ks, ... of row i
__device__ __forceinline__ void row_current(const int32_t* fcol, const double2* fgb, const double2* v, int k0, int k1, int ks, double& ire, double& iim) {
    for (int k = k0; k < k1; k += ks) {
        const double2 y = fgb[k], x = v[fcol[k]];
        ire += y.x * x.x - y.y * x.y;
        iim += y.y * x.x + y.x * x.y;
    }
}
__device__ __forceinline__ void recover_row(const RecoverArgs& A, size_t o, int i, const double2* v, bool warp) {
    const int k0 = A.fptr[i], k1 = A.fptr[i + 1], lane = threadIdx.x & 31;
    double ire = 0.0, iim = 0.0;
    row_current(A.fcol, A.fgb, v, warp ? k0 + lane : k0, k1, warp ? 32 : 1, ire, iim);
    if (warp) { ire = warp_sum(ire); iim = warp_sum(iim); if (lane) return; }
    const double2 vi = v[i];
    A.p_inj[o + i] = vi.x * ire + vi.y * iim;
    A.q_inj[o + i] = vi.y * ire - vi.x * iim;
}

__global__ void k_recover(const RecoverArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int b = blockIdx.x;
    const size_t o = (size_t)b * A.n_bus;
    double2* v = A.v_in_smem ? reinterpret_cast<double2*>(smem) : reinterpret_cast<double2*>(A.work + (size_t)b * A.work_stride);
    for (int i = threadIdx.x; i < A.n_bus; i += blockDim.x) {
        double sn, cs; sincos(A.va[o + i], &sn, &cs);
        const double m = A.vm[o + i];
        v[i] = make_double2(m * cs, m * sn);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < A.n_bus; i += blockDim.x)
        if (A.fptr[i + 1] - A.fptr[i] <= kLongRow) recover_row(A, o, i, v, false);
    for (int r = threadIdx.x >> 5; r < A.n_long; r += blockDim.x >> 5) recover_row(A, o, A.long_rows[r], v, true);
}

// the same as two launches over all (scenario, bus) pairs with V in the scenarios' workspace slices: for grids whose V takes
// most of an SM's shared memory (one CTA per SM, a batch of a few hundred scenarios in two waves)
// (the row pass serves kRecS scenarios per thread: the Y entries of a row are loaded once for all of them, and their gathers
// are independent loads in flight together)
constexpr int kRecS = 4;
template <int kPass>
__global__ void k_recover_flat(const RecoverArgs A) {
    if (kPass == 0) {
        const size_t total = (size_t)A.batch * A.n_bus;
        for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
            const int b = (int)(idx / A.n_bus), i = (int)(idx - (size_t)b * A.n_bus);
            double2* v = reinterpret_cast<double2*>(A.work + (size_t)b * A.work_stride);
            double sn, cs; sincos(A.va[idx], &sn, &cs);
            const double m = A.vm[idx];
            v[i] = make_double2(m * cs, m * sn);
        }
        return;
    }
    const int nbg = (A.batch + kRecS - 1) / kRecS;                       // groups of kRecS scenarios
    const size_t total = (size_t)nbg * A.n_bus;
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int bg = (int)(idx / A.n_bus), i = (int)(idx - (size_t)bg * A.n_bus);
        const int k0 = A.fptr[i], k1 = A.fptr[i + 1];
        if (k1 - k0 > kLongRow) continue;
        const double2* v[kRecS];
        double ire[kRecS], iim[kRecS];
#pragma unroll
        for (int q = 0; q < kRecS; ++q) {
            const int b = min(bg * kRecS + q, A.batch - 1);
            v[q] = reinterpret_cast<const double2*>(A.work + (size_t)b * A.work_stride);
            ire[q] = 0.0; iim[q] = 0.0;
        }
        for (int k = k0; k < k1; ++k) {
            const double2 y = A.fgb[k];
            const int j = A.fcol[k];
#pragma unroll
            for (int q = 0; q < kRecS; ++q) {
                const double2 x = v[q][j];
                ire[q] += y.x * x.x - y.y * x.y;
                iim[q] += y.y * x.x + y.x * x.y;
            }
        }
#pragma unroll
        for (int q = 0; q < kRecS; ++q) {
            const int b = bg * kRecS + q;
            if (b < A.batch) {
                const double2 vi = v[q][i];
                A.p_inj[(size_t)b * A.n_bus + i] = vi.x * ire[q] + vi.y * iim[q];
                A.q_inj[(size_t)b * A.n_bus + i] = vi.y * ire[q] - vi.x * iim[q];
            }
        }
    }
    const size_t nw = ((size_t)gridDim.x * blockDim.x) >> 5, tot = (size_t)A.batch * A.n_long;
    for (size_t w = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5; w < tot; w += nw) {
        const int b = (int)(w / A.n_long), r = (int)(w - (size_t)b * A.n_long);
        recover_row(A, (size_t)b * A.n_bus, A.long_rows[r], reinterpret_cast<const double2*>(A.work + (size_t)b * A.work_stride), true);
    }
}

// ---- implicit-layer backward (eqs. 10-16) around the adjoint solve ---------------------------------
// Layer: x = [p_g at PV; Vm at PV and slack] -> y = [p_g, q_g at PV and slack; Vm; theta] through Step 1 (F1 = 0) and
// Step 2 (recovery).  With F = S_calc - S_spec (this repository's sign):
//   pre : g_theta_j = dL/dtheta_j + sum_i [a_i dP_i/dtheta_j + c_i dQ_i/dtheta_j],  g_Vm_j likewise            (eq. 11-13)
//         with a_i = dL/dp_g,i at the slack, c_i = dL/dq_g,i at PV and slack buses (the rows of z2, eq. 5)
//   solve J1^T lambda = [g_theta (non-slack); g_Vm (PQ)]                                                        (eq. 14)
//   post: dL/dp_g,k = dL/dp_g,k + lambda_P,k (PV);  dL/dVm_k = g_Vm_k - sum_i [lambda_P,i dP_i/dVm_k + lambda_Q,i dQ_i/dVm_k]  (eq. 15-16)
// Jacobian entries are evaluated on the fly from Y_bus and V with the Alg. 1 formulas (the rows / columns needed here are
// not part of J1).  One CTA per scenario; V and (P, Q) per bus in shared memory, or in the scenario's workspace slice.
struct LayerArgs {
    int32_t n_bus, batch, in_smem, post;
    const int32_t *fptr, *fcol, *ftpos;      // full Y_bus CSR (bus order) and the position of each entry's transpose
    const double2* fgb;
    const uint8_t* bus_type;
    const double *vm, *va;                   // [batch][n_bus] solved state
    const double *gl_pg, *gl_qg, *gl_vm, *gl_va;   // loss partials w.r.t. the output buffer y
    double *g_va, *g_vm;                     // pre: out (right-hand side of eq. 14 and the Vm part of g_x); post: in
    const double *lam_p, *lam_q;             // post: in
    double *dx_pg, *dx_vm;                   // post: out
    char* work; int64_t work_stride;
    const int32_t* long_rows; int32_t n_long;   // buses whose Y_bus row has more than kLongRow entries (served by a whole warp)
};

__device__ __forceinline__ void jac_entry(double2 y, double2 vi, double2 vj, double vmj, double& dP_dth, double& dP_dvm,
                                          double& dQ_dth, double& dQ_dvm) {   // off-diagonal, theta_ij = theta_i - theta_j
    const double a = vi.x * vj.x + vi.y * vj.y, b = vi.y * vj.x - vi.x * vj.y;
    const double u1 = y.x * b - y.y * a, u2 = y.x * a + y.y * b, iv = 1.0 / vmj;
    dP_dth = u1; dP_dvm = u2 * iv; dQ_dth = -u2; dQ_dvm = u1 * iv;
}

// The three passes of k_layer for one bus of scenario b (o = b * n_bus; v, pq, w: the scenario's scratch arrays)
__device__ __forceinline__ void layer_pass_state(const LayerArgs& A, size_t o, int i, double2* v, double2* w) {
    double sn, cs; sincos(A.va[o + i], &sn, &cs);
    const double vm = A.vm[o + i];
    v[i] = make_double2(vm * cs, vm * sn);
    const int ti = A.bus_type[i];
    if (!A.post) w[i] = make_double2(ti == 2 ? A.gl_pg[o + i] : 0.0, ti != 0 ? A.gl_qg[o + i] : 0.0);   // rows of z2: P at the slack, Q at PV / slack
    else         w[i] = make_double2(ti != 2 ? A.lam_p[o + i] : 0.0, ti == 0 ? A.lam_q[o + i] : 0.0);   // rows of J1: P non-slack, Q at PQ
}
// (warp = true: the row is served by a whole warp, see kLongRow)
__device__ __forceinline__ void layer_pass_injections(const LayerArgs& A, int i, const double2* v, double2* pq, bool warp) {
    const int k0 = A.fptr[i], k1 = A.fptr[i + 1], lane = threadIdx.x & 31;
    double ire = 0.0, iim = 0.0;
    row_current(A.fcol, A.fgb, v, warp ? k0 + lane : k0, k1, warp ? 32 : 1, ire, iim);
    if (warp) { ire = warp_sum(ire); iim = warp_sum(iim); if (lane) return; }
    pq[i] = make_double2(v[i].x * ire + v[i].y * iim, v[i].y * ire - v[i].x * iim);
}
__device__ __forceinline__ void layer_pass_columns(const LayerArgs& A, size_t o, int j, const double2* v, const double2* pq, const double2* w, bool warp) {
    const int tj = A.bus_type[j], lane = threadIdx.x & 31;
    const double vmj = A.vm[o + j];
    const int k0 = warp ? A.fptr[j] + lane : A.fptr[j], k1 = A.fptr[j + 1], ks = warp ? 32 : 1;
    double a1 = 0.0, a2 = 0.0;             // the two column sums (theta_j / Vm_j), rows weighted by w
    if (!A.post) {
        for (int k = k0; k < k1; k += ks) {
            const int i = A.fcol[k], ti = A.bus_type[i];
            if (ti == 0) continue;                                   // rows of z2 sit at PV and slack buses only
            const double ai = w[i].x, ci = w[i].y;
            double dP_dth, dP_dvm, dQ_dth, dQ_dvm;
            if (i == j) {
                const double2 y = A.fgb[k], s = pq[i];
                dP_dth = -s.y - y.y * vmj * vmj;  dP_dvm = s.x / vmj + y.x * vmj;
                dQ_dth = s.x - y.x * vmj * vmj;   dQ_dvm = s.y / vmj - y.y * vmj;
            } else jac_entry(A.fgb[A.ftpos[k]], v[i], v[j], vmj, dP_dth, dP_dvm, dQ_dth, dQ_dvm);
            a1 += ai * dP_dth + ci * dQ_dth;
            a2 += ai * dP_dvm + ci * dQ_dvm;
        }
    } else if (A.post == 2) {
        // residual of eq. 14 in FP64, r = g - J1^T lambda (here gl_va / gl_vm = g, output g_va / g_vm = r): column
        // theta_j of every non-slack bus, column Vm_j of every PQ bus; rows P_i (non-slack), Q_i (PQ)
        if (tj != 2)
            for (int k = k0; k < k1; k += ks) {
                const int i = A.fcol[k], ti = A.bus_type[i];
                if (ti == 2) continue;
                const double lp = w[i].x, lq = w[i].y;
                double dP_dth, dP_dvm, dQ_dth, dQ_dvm;
                if (i == j) {
                    const double2 y = A.fgb[k], s = pq[i];
                    dP_dth = -s.y - y.y * vmj * vmj;  dP_dvm = s.x / vmj + y.x * vmj;
                    dQ_dth = s.x - y.x * vmj * vmj;   dQ_dvm = s.y / vmj - y.y * vmj;
                } else jac_entry(A.fgb[A.ftpos[k]], v[i], v[j], vmj, dP_dth, dP_dvm, dQ_dth, dQ_dvm);
                a1 += lp * dP_dth + lq * dQ_dth;
                a2 += lp * dP_dvm + lq * dQ_dvm;
            }
    } else {
        if (tj != 0)
            for (int k = k0; k < k1; k += ks) {
                const int i = A.fcol[k];
                const double lp = w[i].x, lq = w[i].y;
                double dP_dth, dP_dvm, dQ_dth, dQ_dvm;
                if (i == j) {
                    const double2 y = A.fgb[k], s = pq[i];
                    dP_dvm = s.x / vmj + y.x * vmj;  dQ_dvm = s.y / vmj - y.y * vmj;
                } else jac_entry(A.fgb[A.ftpos[k]], v[i], v[j], vmj, dP_dth, dP_dvm, dQ_dth, dQ_dvm);
                a2 += lp * dP_dvm + lq * dQ_dvm;
            }
    }
    if (warp) { a1 = warp_sum(a1); a2 = warp_sum(a2); if (lane) return; }
    if (!A.post) {
        A.g_va[o + j] = tj != 2 ? A.gl_va[o + j] + a1 : 0.0;
        A.g_vm[o + j] = A.gl_vm[o + j] + a2;
    } else if (A.post == 2) {
        A.g_va[o + j] = tj != 2 ? A.gl_va[o + j] - a1 : 0.0;
        A.g_vm[o + j] = tj == 0 ? A.gl_vm[o + j] - a2 : 0.0;
    } else {
        A.dx_vm[o + j] = tj != 0 ? A.g_vm[o + j] - a2 : 0.0;
        A.dx_pg[o + j] = tj == 1 ? A.gl_pg[o + j] + A.lam_p[o + j] : 0.0;
    }
}

// one CTA per scenario; scratch in shared memory, or (grids whose 48 n_bus bytes do not fit) in the scenario's workspace slice.
// (The three passes as launches over all (scenario, bus) pairs, in one piece or in L2-sized chunks of scenarios, were measured on
// config 5: 0.34 ms per call and more against 0.27 -- the row passes re-read the Y entries for every scenario either way.)
__global__ void k_layer(const LayerArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int b = blockIdx.x, nb = A.n_bus, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const size_t o = (size_t)b * nb;
    double2* v = A.in_smem ? reinterpret_cast<double2*>(smem) : reinterpret_cast<double2*>(A.work + (size_t)b * A.work_stride);
    double2* pq = v + nb;
    double2* w = pq + nb;                  // per bus i: the two row weights the transposed products gather (coalesced here)
    for (int i = threadIdx.x; i < nb; i += blockDim.x) layer_pass_state(A, o, i, v, w);
    __syncthreads();
    for (int i = threadIdx.x; i < nb; i += blockDim.x)
        if (A.fptr[i + 1] - A.fptr[i] <= kLongRow) layer_pass_injections(A, i, v, pq, false);
    for (int r = warp; r < A.n_long; r += nwarp) layer_pass_injections(A, A.long_rows[r], v, pq, true);
    __syncthreads();
    for (int j = threadIdx.x; j < nb; j += blockDim.x)
        if (A.fptr[j + 1] - A.fptr[j] <= kLongRow) layer_pass_columns(A, o, j, v, pq, w, false);
    for (int r = warp; r < A.n_long; r += nwarp) layer_pass_columns(A, o, A.long_rows[r], v, pq, w, true);
}

// lambda += correction (iterative refinement of the adjoint, sable_adjoint_refined)
__global__ void k_add2(double* xp, double* xq, const double* dp, const double* dq, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        xp[i] += dp[i]; xq[i] += dq[i];
    }
}

// ---- debug: state from caller's (vm, va), mismatch / Jacobian / refactor at that state ---------------------------
struct DebugArgs {
    DevTemplate t;
    int32_t batch, what;              // what: 0 mismatch, 1 jacobian, 2 refactor only (factors kept for k_linsolve)
    const double *p_spec, *q_spec, *vm, *va;
    double *f_p, *f_q, *norm, *diag, *pairs;
    char* factors; char* work; int64_t fac_stride, work_stride;
    const double* zeros;              // [n_bus] zeros: stands in for absent p_spec / q_spec
    int32_t* pivot;                   // [batch] tiny-pivot flags (what = 2), or nullptr
};

template <typename T>
__global__ void k_debug(const DebugArgs A) {
    __shared__ double red[32 * 32];
    __shared__ double scratch[32 * kBigDoubles];
    const DevTemplate& t = A.t;
    const int b = blockIdx.x;
    const Slot<T, 2> s = hbm_slot<T>(t, A.factors, A.fac_stride, A.work, A.work_stride, b);
    const PivotFlag pf{A.pivot ? A.pivot + b : nullptr};
    if (A.pivot && threadIdx.x == 0) A.pivot[b] = 0;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
        const int bus = t.node_bus[m];
        const double vm = A.vm[o + bus], th = A.va[o + bus];
        double sn, cs; sincos(th, &sn, &cs);
        s.set_ma(m, make_double2(vm, th));
        s.set_vv(m, make_double2(vm * cs, vm * sn));
    }
    if (A.what == 1) {                                               // export of J: the fill-in pairs (never written by the walk) read as zero
        const Blk<T> z = {T(0), T(0), T(0), T(0)};
        for (int p = threadIdx.x; p < t.n_pair; p += blockDim.x) s.stUL(p, z, z);
    }
    __syncthreads();
    const double r = slot_max_nan(stage_mismatch<T, 2>(t, s, A.p_spec ? A.p_spec + o : A.zeros, A.q_spec ? A.q_spec + o : A.zeros, true, 0, pf, Team{0, 1}), red, 0);
    if (A.what == 0) {
        for (int m = threadIdx.x; m <= t.n_node; m += blockDim.x) {
            const int bus = t.node_bus[m];
            const double2 f = m < t.n_node ? s.rh(m) : make_double2(0.0, 0.0);
            A.f_p[o + bus] = m < t.n_node ? -f.x : 0.0;
            A.f_q[o + bus] = m < t.n_node ? -f.y : 0.0;
        }
        if (threadIdx.x == 0) A.norm[b] = r;
        return;
    }
    stage_fill_pairs<T, 2>(t, s, threadIdx.x, blockDim.x);
    __syncthreads();
    if (A.what == 1) {
        for (int m = threadIdx.x; m < t.n_node; m += blockDim.x) {
            const Blk<T> d = s.ldD(m);
            double* o4 = A.diag + ((size_t)b * t.n_node + m) * 4;
            o4[0] = double(d.a); o4[1] = double(d.b); o4[2] = double(d.c); o4[3] = double(d.d);
        }
        for (int p = threadIdx.x; p < t.n_pair; p += blockDim.x) {
            Blk<T> U, L;
            s.ldUL(p, U, L);
            double* o8 = A.pairs + ((size_t)b * t.n_pair + p) * 8;
            o8[0] = double(U.a); o8[1] = double(U.b); o8[2] = double(U.c); o8[3] = double(U.d);
            o8[4] = double(L.a); o8[5] = double(L.b); o8[6] = double(L.c); o8[7] = double(L.d);
        }
        return;
    }
    BlobRing ring = no_ring(t);
    stage_factor_forward<T, 2, true, false, false, false>(t, s, t.level, ring, pf, scratch, Team{0, 1});
}

}  // namespace sable
