// The fused persistent Newton-Raphson kernel: a CTA takes groups of G scenarios from an atomic queue and runs the whole
// NR loops of a group's scenarios in lockstep, with no host round trip; a scenario that converged (or stopped) is no
// longer evaluated -- the per-scenario convergence masking.  Launched from sable_capi.cu.
#pragma once
#include "sable_stages.cuh"
#include "sable_front.cuh"

namespace sable {

struct SolveArgs {
    DevTemplate t;
    int32_t batch, max_it, keep, trash_grp;               // trash_grp: spare group of the workspace (finished slots run along on it)
    double tol;
    const double *p_spec, *q_spec, *v_set, *vm0, *va0;    // [batch][n_bus]
    double *vm, *va, *final_norm;
    int32_t* iterations;
    uint8_t* converged;
    int32_t* pivot;           // [batch] tiny-pivot flags: bit 0 = seen in some refactorisation of the scenario, bit 1 = in the last one
    char* factors;            // [groups + 1][fac_stride << gsh] bytes, group-interleaved (sable_device.cuh)
    char* work;               // [groups + 1][work_stride << gsh] bytes
    int64_t fac_stride, work_stride;
    int32_t gsh;                                           // slots per CTA = 1 << gsh
    int32_t csz;                                           // CTAs per team (cluster size); 1 = every CTA works alone
    double* team_red;                                      // [teams][csz][G] per-slot norm partials of the CTAs of a team
    int32_t ring_r, ring_slot, first_staged;               // level-blob ring: slots, bytes per slot, first streamed level
    int32_t front_k, front_f0, front_level;                // dense top front (sable_front.cuh): K nodes from f0 = levels >= front_level; 0 = off
    int32_t big_off;                                       // byte offset of the big-target scratch in dynamic shared memory
    int32_t slot_off;                                      // on-chip placement: byte offset of the slots in dynamic shared memory
    int64_t front_off;                                     // HBM placement: byte offset of the front in dynamic shared memory
    LevelDesc front;                                       // assembly lists of the front
    unsigned long long* tim;  // optional cycle counters (sable_debug_timing), else nullptr
    int32_t* queue;           // persistent-kernel scenario counter
    int32_t* status;          // staged mode: [batch] 0 = active, 1 = converged, 2 = stopped
    int32_t* it;              // staged mode: [batch]
    int32_t* active;          // staged mode: [max_it + 2] scenarios still active after each mismatch pass
    int32_t stage_it;         // staged mode: index of this mismatch pass
    // inner refinement of the forward linear solve (sable_options.ir_sweeps > 0; staged mode, FP32 factors): the solve stage
    // leaves the step in rh instead of applying it, and the refinement works on bus-order arrays [batch][n_bus]
    int32_t ir;
    double2* ir_v;            // rectangular voltages of the current iterate
    double *ir_vm, *ir_dzp, *ir_dzq;   // |V|; the step: theta part (non-slack buses), Vm part (PQ buses), zero elsewhere
    const int32_t* ir_bus_node;        // [n_bus] node of each bus (slack -> n_node)
};

constexpr int kRedBytes = 32 * 32 * 8;                      // per-slot norm reduction scratch: 32 warps x 32 slots
constexpr int kSmemHeader = kRedBytes + 128 + 8 * kMaxRing; // + slot bookkeeping + ring mbarriers
__host__ __device__ inline int64_t align16(int64_t x) { return (x + 15) & ~int64_t(15); }
template <typename T> __host__ __device__ inline int64_t fac_bytes(int n_node, int n_pair) { return (int64_t)(n_node + 2 * (int64_t)n_pair) * 4 * sizeof(T); }
__host__ __device__ inline int64_t work_bytes(int n_node) { return 3 * (int64_t)(n_node + 1) * 16; }
__host__ __device__ inline int64_t big_bytes(int threads, int gsh) { return ((int64_t)(threads >> 5) * kBigDoubles * 8) << gsh; }
// dynamic shared memory: header, level descriptors, blob ring, big-target scratch, then (on-chip placement) the slots
__host__ __device__ inline int64_t smem_fixed(int n_level, int ring_bytes, int big) {
    return kSmemHeader + align16((int64_t)n_level * (int64_t)sizeof(LevelDesc)) + align16(ring_bytes) + align16(big);
}
template <typename T> __host__ __device__ inline int64_t smem_need(int n_node, int n_pair, int n_level, int ring_bytes, int big, int gsh, bool on_chip) {
    int64_t b = smem_fixed(n_level, ring_bytes, big);
    if (on_chip) b += (work_bytes(n_node) + fac_bytes<T>(n_node, n_pair)) << gsh;
    return b;
}

// shared-memory part of a slot view (fixed for the lifetime of the CTA) and the CTA-uniform offsets of the HBM arrays
template <typename T, int kP>
__device__ __forceinline__ Slot<T, kP> carve(unsigned char* smem, int64_t slot_off, int n_node, int n_pair, int gsh, int g) {
    Slot<T, kP> s;
    const unsigned ns = (unsigned)(((size_t)(n_node + 1) * 16) << gsh), nd = (unsigned)(((size_t)n_node * 4 * sizeof(T)) << gsh);
    const unsigned np = (unsigned)(((size_t)n_pair * 4 * sizeof(T)) << gsh);
    s.sb = reinterpret_cast<char*>(smem) + slot_off + g * 16;
    s.so_ma = ns; s.so_rh = 2 * ns; s.so_dg = 3 * ns; s.so_pu = s.so_dg + nd; s.so_pl = s.so_pu + np;
    s.gf = s.gw = nullptr;
    s.go_pu = Slot<T, kP>::kPairRec ? ((nd + 31u) & ~31u) : nd;      // pair records (FP32 factors in HBM) are 32-byte aligned
    s.go_pl = s.go_pu + np; s.go_ma = ns; s.go_rh = 2 * ns;
    s.gsh = gsh; s.gpx = 0;
#ifdef SABLE_BOUNDS
    s.nn_ = n_node; s.np_ = n_pair;
#endif
    return s;
}
// HBM part: the slices of scenario b's group (b >> gsh), offset to lane b & (G - 1); strides are per scenario
template <typename T, int kP>
__device__ __forceinline__ void bind(Slot<T, kP>& s, char* factors, int64_t fac_stride, char* work, int64_t work_stride, int b) {
    const int gsh = s.gsh;
    const size_t grp = (size_t)(b >> gsh), lane16 = (size_t)(b & ((1 << gsh) - 1)) * 16;
    s.gf = factors + ((grp * (size_t)fac_stride) << gsh) + (size_t)(b & ((1 << gsh) - 1)) * (4 * sizeof(T));   // whole blocks interleave
    s.gw = work + ((grp * (size_t)work_stride) << gsh) + lane16;
    s.gpx = Slot<T, kP>::kPairRec ? (unsigned)lane16 : 0u;     // pair records are 32 bytes wide: 16 more per lane than the blocks
}

template <typename T, int kP>
__device__ __forceinline__ void scen_init(const SolveArgs& A, const Slot<T, kP>& s, int b, int tsub, int nsub) {
    const DevTemplate& t = A.t;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = tsub; m <= t.n_node; m += nsub) {       // PAPER.md:287 flat start unless vm0/va0 given
        const int bus = t.node_bus[m];
        const bool pq = m < t.n_node && t.node_pq[m];
        const double vm = pq ? (A.vm0 ? A.vm0[o + bus] : 1.0) : A.v_set[o + bus];
        const double th = A.va0 ? A.va0[o + bus] : 0.0;
        double sn, cs; sincos(th, &sn, &cs);
        s.set_ma(m, make_double2(vm, th));
        s.set_vv(m, make_double2(vm * cs, vm * sn));
    }
    if (tsub == 0) A.pivot[b] = 0;
}

template <typename T, int kP>
__device__ __forceinline__ void scen_output(const SolveArgs& A, const Slot<T, kP>& s, int b, int it, bool conv, double r, int tsub, int nsub) {
    const DevTemplate& t = A.t;
    const size_t o = (size_t)b * t.n_bus;
    for (int m = tsub; m <= t.n_node; m += nsub) {
        const int bus = t.node_bus[m];
        const double2 a = s.ma(m);
        A.vm[o + bus] = a.x; A.va[o + bus] = a.y;
    }
    if (tsub == 0) {
        A.iterations[b] = conv ? it : A.max_it;
        A.converged[b] = conv ? 1 : 0;
        if (A.final_norm) A.final_norm[b] = r;
    }
}

// kept factors (reading 16): the on-chip factors of J1 at the final iterate go to the
// scenario's HBM slice (same order dg | pu | pl, same interleaving)
template <typename T, int kP>
__device__ __forceinline__ void store_factors(const DevTemplate& t, const Slot<T, kP>& s, int tsub, int nsub) {
    // dg | pu | pl are contiguous block arrays in both memories: block i of the shared copy goes to block i of the HBM slice
    Slot<T, 2> h = carve<T, 2>(nullptr, 0, t.n_node, t.n_pair, s.gsh, 0);    // the HBM view of the same slot
    h.sb = nullptr; h.gf = s.gf; h.gw = s.gw;
    h.gpx = Slot<T, 2>::kPairRec ? (unsigned)((threadIdx.x & ((1 << s.gsh) - 1)) * 16) : 0u;
    for (int i = tsub; i < t.n_node; i += nsub) h.stD(i, s.ldD(i));
    for (int p = tsub; p < t.n_pair; p += nsub) h.stUL(p, s.ldU(p), s.ldL(p));
}

__device__ __forceinline__ int pop_group(const SolveArgs& A) {
    const int v = atomicAdd(A.queue, 1);
    return v < ((A.batch + (1 << A.gsh) - 1) >> A.gsh) ? v : -1;
}

// Loop convention, per slot:
//   it = 0; loop { r = ||F1||inf; if r <= tol: converged; if it == max_it or r not finite: stop; solve; update; ++it }
// A CTA takes one GROUP of G consecutive scenarios at a time from the atomic queue (slot g serves scenario
// group * G + g, whose HBM slices are interleaved with the rest of its group) and advances its slots in lockstep; a slot
// that has finished stops being evaluated (its lanes run along and write nothing that is read) until the group is done.
// Register budgets: on chip 1 CTA of up to 512 threads (up to 128 registers); HBM placement kCtas CTAs per SM of up to
// kThreads threads each.
template <typename T, int kP, int kThreads, int kCtas>
__global__ void __launch_bounds__(kThreads, kCtas) k_nr_fused(const SolveArgs A) {
    extern __shared__ __align__(16) unsigned char smem[];
    const DevTemplate& t = A.t;
    // team of CTAs (cluster) serving one group together: HBM placement only; every CTA of a team runs the same control flow
    const Team tm{kP == 2 && A.csz > 1 ? cluster_ctarank() : 0, kP == 2 && A.csz > 1 ? A.csz : 1};
    const int team = blockIdx.x / tm.csz, n_teams = gridDim.x / tm.csz;
    const int gsh = A.gsh, G = 1 << gsh, g = threadIdx.x & (G - 1);
    const int tsub_c = threadIdx.x >> gsh, nsub_c = blockDim.x >> gsh;               // lanes of this CTA (front, on-chip copies)
    const int tsub = tm.rank * nsub_c + tsub_c, nsub = nsub_c * tm.csz;              // lanes of the team (wide passes)
    double* red = reinterpret_cast<double*>(smem);
    int* s_b = reinterpret_cast<int*>(smem + kRedBytes);
    LevelDesc* lv = reinterpret_cast<LevelDesc*>(smem + kSmemHeader);
    for (int i = threadIdx.x; i < t.n_level; i += blockDim.x) lv[i] = t.level[i];
    double* scratch = reinterpret_cast<double*>(smem + A.big_off);
    Slot<T, kP> s = carve<T, kP>(smem, A.slot_off, t.n_node, t.n_pair, gsh, g);
    Front<T> F = carve_front<T>(smem, A.front_off, A.front_k, A.front_f0, gsh, g);
    BlobRing ring;
    ring.slots = reinterpret_cast<char*>(smem) + kSmemHeader + align16((int64_t)t.n_level * (int64_t)sizeof(LevelDesc));
    ring.mbar = reinterpret_cast<unsigned long long*>(smem + kRedBytes + 128);
    ring.gblob = t.blob; ring.lv = lv; ring.R = A.ring_r; ring.slot_bytes = A.ring_slot;
    ring.first = A.first_staged; ring.n_level = t.n_level;
    ring.on = kP == 0 && A.ring_r > 0;
#ifdef SABLE_TIMING_ALL
    ring.tim = blockIdx.x == 0 ? A.tim : nullptr;
#else
    ring.tim = (kP == 0 && blockIdx.x == 0) ? A.tim : nullptr;   // HBM-placement kernels: counters compiled out (registers)
#endif
    long long tk = clock64();
    __syncthreads();                                       // lv[] complete before the producer reads it
    ring.start();
    const double kInf = __longlong_as_double(0x7ff0000000000000LL);
    int b = -1, it = 0, next_grp = team;
    bool fin = false;
    PivotFlag pf{nullptr};
    auto to_trash = [&]() {
        b = -1; pf.w = nullptr;
        bind<T, kP>(s, A.factors, A.fac_stride, A.work, A.work_stride, (A.trash_grp << gsh) + g);
    };
    auto any_slot = [&](bool mine) {                       // CTA-uniform OR over the slots (team-uniform: the state is replicated); two barriers
        __syncthreads();
        if (threadIdx.x < G) s_b[threadIdx.x] = mine ? 1 : 0;
        __syncthreads();
        bool any = false;
        for (int x = 0; x < G; ++x) any |= s_b[x] != 0;
        return any;
    };
    for (;;) {
        if (b >= 0 && tsub == 0) atomicAnd(pf.w, 1);       // bit 1 = "in the last refactorisation": cleared before each one
        if (tm.csz > 1) team_sync(tm);                     // the update of the last trip (all CTAs) before this trip's mismatch
        if (!any_slot(b >= 0)) {                           // group done: take the next one
            int grp;
            if (tm.csz > 1) {                              // teams: static assignment (team t serves groups t, t + n_teams, ...)
                grp = next_grp < ((A.batch + G - 1) >> gsh) ? next_grp : -1;
                next_grp += n_teams;
            } else {
                __syncthreads();
                if (threadIdx.x == 0) s_b[0] = pop_group(A);
                __syncthreads();
                grp = s_b[0];
            }
            if (grp < 0) { ring.drain(); break; }
            const int bb = (grp << gsh) + g;
            bind<T, kP>(s, A.factors, A.fac_stride, A.work, A.work_stride, bb);
            b = bb < A.batch ? bb : -1;
            it = 0; fin = false;
            if (b < 0) to_trash();
            else { pf.w = A.pivot + b; scen_init<T, kP>(A, s, b, tsub, nsub); }
            team_sync(tm);
        }
        ring.tick(4 * t.n_level + 2, tk);                  // group bookkeeping + init
        {
            const size_t row = (size_t)(b >= 0 ? b : 0) * t.n_bus;
            const double loc = stage_mismatch<T, kP>(t, s, A.p_spec + row, A.q_spec + row, b >= 0, lv[0].m1, pf, tm);
            double r = slot_max_nan(loc, red, gsh);
            if (tm.csz > 1) {                              // combine the CTAs' per-slot norms through the team's scratch words
                double* tr = A.team_red + (size_t)team * tm.csz * G;
                if (threadIdx.x < G) tr[tm.rank * G + g] = r;
                team_sync(tm);
                r = tr[g];
                for (int k = 1; k < tm.csz; ++k) r = nan_max(r, tr[k * G + g]);
            }
            ring.tick(4 * t.n_level + 3, tk);              // mismatch + norm
            if (b >= 0) {
                bool done = false, conv = false;
                if (r <= A.tol) { done = true; conv = true; }
                else if (it == A.max_it || !(fabs(r) < kInf)) done = true;
                if (done) {
                    scen_output<T, kP>(A, s, b, it, conv, r, tsub, nsub);
                    if (A.keep) fin = true;
                    else to_trash();
                }
            }
        }
        if (!any_slot(b >= 0)) continue;                   // every slot finished (and no factors to keep)
        // a2 happened inside the mismatch walk (stage_mismatch), or happens here as a pass over the pairs (FP32 pair records);
        // either way the pairs with a Y entry hold J afterwards and the fill-in pairs nothing yet
        stage_fill_pairs<T, kP>(t, s, tsub, nsub);
        if (kP == 2 && A.front_k > 0) front_zero<T>(F, tsub_c, nsub_c);
        team_sync(tm);
        ring.tick(4 * t.n_level, tk);                      // decision + output + Jacobian fill
        if (kP == 2) {
            // HBM placement: the levels below the dense top front level by level (all of them if there is no front:
            // front_level = n_level), the front itself as one dense block in shared memory (sable_front.cuh; a CTA working
            // alone only)
            stage_factor_forward<T, kP, true, true, false, true, false>(t, s, lv, ring, pf, scratch, tm, A.front_level);
            if (A.front_k > 0) {
                tk = clock64();
                front_assemble<T, kP, true>(t, s, F, A.front, pf, scratch, tsub_c, nsub_c);
                ring.tick(3, tk);
                front_factor<T, true>(F, pf, tsub_c, nsub_c);
                ring.tick(7, tk);
            }
            if (any_slot(b >= 0 && !fin)) {                // a trip that only refactors for kept factors needs no solve
                if (A.front_k > 0) { front_backward<T, kP>(s, F, tsub_c, nsub_c); ring.tick(11, tk); }
                stage_backward<T, kP, false, false>(t, s, lv, ring, tm, A.front_level);
                stage_update<T, kP>(t, s, tsub, nsub);
            }
            if (fin && A.front_k > 0) front_store<T, kP>(t, s, F, A.front, tsub_c, nsub_c);
        } else {
            stage_factor_forward<T, kP, true, true, false, true>(t, s, lv, ring, pf, scratch, tm);
            if (any_slot(b >= 0 && !fin)) {
                stage_backward<T, kP, false>(t, s, lv, ring, tm);
                stage_update<T, kP>(t, s, tsub, nsub);
            } else ring.skip_sweep();
        }
        if (ring.tim && threadIdx.x == 0) { ring.tim[4 * t.n_level + 1] += 1; tk = clock64(); }   // trips
        if (b >= 0 && !fin) ++it;
        if (fin) {
            if (kP == 0) store_factors<T, kP>(t, s, tsub, nsub);
            fin = false; to_trash();                       // the kept factors stay untouched: run along on the spare group
        }
    }
    if (tm.csz > 1) team_sync(tm);                         // no CTA of a cluster exits while a peer may still wait on it
}

}  // namespace sable
