/*
 * sable_oracle.c -- CPU FP64 oracle for the batched Newton-Raphson AC power flow + adjoint of SABLE
 * (arxiv/paper_2606_07099).  TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs.  It shares no code with the CUDA path
 * (paper_2606_07099_b200/) and the product never calls it.
 *
 * Plain, slow, written to be checked against the paper by eye.  Citations are PAPER.md lines.
 *   - net injections / mismatch:  PAPER.md:55 (S_spec = gen - load), :84 eq. (6) F1 = [dP_{B\R}; dQ_D],
 *     real form PAPER.md:201-207 (V_re, V_im, I_re, I_im).  Sign: F = S_calc - S_spec (reading 5;
 *     the Newton step is the same as with the paper's spec - calc, lambda flips sign).
 *   - Jacobian J1 = d[P_{B\R}; Q_D] / d[theta_{B\R}; Vm_D]: eq. (8).  Algorithm 1's entry
 *     formulas are lost in the extraction; the textbook polar-form entries are used
 *     (reading 4) and pinned by finite differences and the complex-matrix identities in tests/.
 *   - Newton step J1 dz = -F1, z += dz: eq. (7).  Flat start PAPER.md:287.  tol 1e-8: :277.
 *   - adjoint J1^T lambda = g at the converged point: eq. (14).
 *   - mixed precision (sanity only): J1 and -F1 rounded to FP32, solve in FP32, dz promoted: PAPER.md:255.
 *
 * Unknown order z = [theta_i, i non-slack ascending; Vm_i, i PQ ascending]; equation order
 * F = [P_i, i non-slack; Q_i, i PQ].  The boundary uses full-bus arrays, so this order is private.
 *
 * Linear solves: dense LU with partial pivoting (method 0) or a textbook right-looking sparse row
 * elimination with partial pivoting, columns taken in ascending-degree order (method 1).  Both are
 * "parity pinned": tests/ check them against each other, against numpy/scipy solves and by residual.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PQ_BUS 0
#define PV_BUS 1
#define SLACK_BUS 2

/* ----------------------------------------------------------------------------------------------- */
/* Y_bus from a branch list (pi-model, no taps / shifters / shunts: DESIGN.md reading 14).
 * Branch (f,t) with series y = 1/(r+jx) and total charging b:
 *   Y_ff += y + jb/2, Y_tt += y + jb/2, Y_ft -= y, Y_tf -= y.
 * Output: CSR with sorted columns, duplicates merged, every diagonal present.
 * Call once with row_ptr/col/g/bb == NULL to get nnz, then again with buffers.  Returns nnz. */
typedef struct { int r, c; double g, b; } trip_t;
static int trip_cmp(const void* a, const void* b) {
    const trip_t* x = (const trip_t*)a; const trip_t* y = (const trip_t*)b;
    if (x->r != y->r) return x->r < y->r ? -1 : 1;
    if (x->c != y->c) return x->c < y->c ? -1 : 1;
    return 0;
}
int oracle_ybus(int n_bus, int n_br, const int* f, const int* t, const double* r, const double* x,
                const double* b, int* row_ptr, int* col, double* g, double* bb)
{
    int m = 4 * n_br + n_bus, k, nnz = 0;
    trip_t* T = (trip_t*)malloc(sizeof(trip_t) * (size_t)m);
    int p = 0;
    for (k = 0; k < n_bus; ++k) { T[p].r = k; T[p].c = k; T[p].g = 0; T[p].b = 0; ++p; }
    for (k = 0; k < n_br; ++k) {
        double den = r[k] * r[k] + x[k] * x[k];
        double ys_g = r[k] / den, ys_b = -x[k] / den;          /* 1/(r+jx) */
        T[p].r = f[k]; T[p].c = f[k]; T[p].g = ys_g;  T[p].b = ys_b + 0.5 * b[k]; ++p;
        T[p].r = t[k]; T[p].c = t[k]; T[p].g = ys_g;  T[p].b = ys_b + 0.5 * b[k]; ++p;
        T[p].r = f[k]; T[p].c = t[k]; T[p].g = -ys_g; T[p].b = -ys_b; ++p;
        T[p].r = t[k]; T[p].c = f[k]; T[p].g = -ys_g; T[p].b = -ys_b; ++p;
    }
    qsort(T, (size_t)m, sizeof(trip_t), trip_cmp);
    if (row_ptr) memset(row_ptr, 0, sizeof(int) * (size_t)(n_bus + 1));
    for (k = 0; k < m; ) {
        int j = k; double sg = 0, sb = 0;
        while (j < m && T[j].r == T[k].r && T[j].c == T[k].c) { sg += T[j].g; sb += T[j].b; ++j; }
        if (row_ptr) { col[nnz] = T[k].c; g[nnz] = sg; bb[nnz] = sb; row_ptr[T[k].r + 1]++; }
        ++nnz; k = j;
    }
    if (row_ptr) for (k = 0; k < n_bus; ++k) row_ptr[k + 1] += row_ptr[k];
    free(T);
    return nnz;
}

/* ----------------------------------------------------------------------------------------------- */
/* Calculated injections, PAPER.md:201-207:
 *   V_re = Vm cos(th), V_im = Vm sin(th); I_re = G V_re - B V_im, I_im = B V_re + G V_im;
 *   P = V_re I_re + V_im I_im,  Q = V_im I_re - V_re I_im     (S = V conj(I)). */
void oracle_injections(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                       const double* vm, const double* va, double* P, double* Q)
{
    int i, k;
    for (i = 0; i < n_bus; ++i) {
        double ire = 0, iim = 0;
        for (k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
            int j = col[k];
            double vre = vm[j] * cos(va[j]), vim = vm[j] * sin(va[j]);
            ire += g[k] * vre - bb[k] * vim;
            iim += bb[k] * vre + g[k] * vim;
        }
        {
            double vre = vm[i] * cos(va[i]), vim = vm[i] * sin(va[i]);
            P[i] = vre * ire + vim * iim;
            Q[i] = vim * ire - vre * iim;
        }
    }
}

/* index maps: th_idx[i] = row/col of (P_i, theta_i) or -1 at the slack; vm_idx[i] = row/col of
 * (Q_i, Vm_i) or -1 off PQ buses.  Returns n = n_PV + 2 n_PQ (J1 is square). */
int oracle_index_maps(int n_bus, const uint8_t* bus_type, int* th_idx, int* vm_idx)
{
    int i, n_th = 0, n_vm = 0;
    for (i = 0; i < n_bus; ++i) th_idx[i] = (bus_type[i] != SLACK_BUS) ? n_th++ : -1;
    for (i = 0; i < n_bus; ++i) vm_idx[i] = (bus_type[i] == PQ_BUS) ? n_th + n_vm++ : -1;
    return n_th + n_vm;
}

/* F1 = [P_i - P_spec,i (non-slack); Q_i - Q_spec,i (PQ)]; returns the unscaled inf-norm.
 * A NaN anywhere makes the norm NaN. */
double oracle_mismatch(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                       const uint8_t* bus_type, const double* p_spec, const double* q_spec,
                       const double* vm, const double* va, const int* th_idx, const int* vm_idx,
                       double* F, double* P, double* Q)
{
    int i; double nrm = 0;
    oracle_injections(n_bus, row_ptr, col, g, bb, vm, va, P, Q);
    for (i = 0; i < n_bus; ++i) {
        if (th_idx[i] >= 0) { double v = P[i] - p_spec[i]; F[th_idx[i]] = v; if (!(fabs(v) <= nrm)) nrm = fabs(v); }
        if (vm_idx[i] >= 0) { double v = Q[i] - q_spec[i]; F[vm_idx[i]] = v; if (!(fabs(v) <= nrm)) nrm = fabs(v); }
    }
    (void)bus_type;
    return nrm;
}

/* J1 as COO triplets (row, col, val); returns the count (<= 4 nnz(Y) + 4 n_bus).
 * Off-diagonal (i != j, Y_ij stored), th_ij = th_i - th_j:
 *   dP_i/dth_j = Vm_i Vm_j (G_ij sin th_ij - B_ij cos th_ij)
 *   dP_i/dVm_j = Vm_i (G_ij cos th_ij + B_ij sin th_ij)
 *   dQ_i/dth_j = -Vm_i Vm_j (G_ij cos th_ij + B_ij sin th_ij)
 *   dQ_i/dVm_j = Vm_i (G_ij sin th_ij - B_ij cos th_ij)
 * Diagonal (uses the calculated P_i, Q_i -- why Alg. 1 takes I_re, I_im as inputs):
 *   dP_i/dth_i = -Q_i - B_ii Vm_i^2      dP_i/dVm_i = P_i / Vm_i + G_ii Vm_i
 *   dQ_i/dth_i =  P_i - G_ii Vm_i^2      dQ_i/dVm_i = Q_i / Vm_i - B_ii Vm_i
 * Every structural entry is emitted even if its value is zero. */
int oracle_jacobian_coo(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                        const double* vm, const double* va, const double* P, const double* Q,
                        const int* th_idx, const int* vm_idx, int* jr, int* jc, double* jv)
{
    int i, k, m = 0;
    for (i = 0; i < n_bus; ++i) {
        double gii = 0, bii = 0;
        for (k = row_ptr[i]; k < row_ptr[i + 1]; ++k) {
            int j = col[k];
            if (j == i) { gii += g[k]; bii += bb[k]; continue; }
            {
                double thij = va[i] - va[j], c = cos(thij), s = sin(thij);
                double a1 = g[k] * s - bb[k] * c, a2 = g[k] * c + bb[k] * s;
                if (th_idx[i] >= 0 && th_idx[j] >= 0) { jr[m] = th_idx[i]; jc[m] = th_idx[j]; jv[m] = vm[i] * vm[j] * a1; ++m; }
                if (th_idx[i] >= 0 && vm_idx[j] >= 0) { jr[m] = th_idx[i]; jc[m] = vm_idx[j]; jv[m] = vm[i] * a2; ++m; }
                if (vm_idx[i] >= 0 && th_idx[j] >= 0) { jr[m] = vm_idx[i]; jc[m] = th_idx[j]; jv[m] = -vm[i] * vm[j] * a2; ++m; }
                if (vm_idx[i] >= 0 && vm_idx[j] >= 0) { jr[m] = vm_idx[i]; jc[m] = vm_idx[j]; jv[m] = vm[i] * a1; ++m; }
            }
        }
        if (th_idx[i] >= 0) { jr[m] = th_idx[i]; jc[m] = th_idx[i]; jv[m] = -Q[i] - bii * vm[i] * vm[i]; ++m; }
        if (th_idx[i] >= 0 && vm_idx[i] >= 0) { jr[m] = th_idx[i]; jc[m] = vm_idx[i]; jv[m] = P[i] / vm[i] + gii * vm[i]; ++m; }
        if (vm_idx[i] >= 0 && th_idx[i] >= 0) { jr[m] = vm_idx[i]; jc[m] = th_idx[i]; jv[m] = P[i] - gii * vm[i] * vm[i]; ++m; }
        if (vm_idx[i] >= 0) { jr[m] = vm_idx[i]; jc[m] = vm_idx[i]; jv[m] = Q[i] / vm[i] - bii * vm[i]; ++m; }
    }
    return m;
}

/* ----------------------------------------------------------------------------------------------- */
/* FP32 emulation for the mixed-precision sanity mode: every +,-,*,/ result is rounded to float
 * (double rounding is innocuous for single operations, 53 >= 2*24+2). */
#define RND(sp, e) ((sp) ? (double)(float)(e) : (e))

/* Dense LU with partial (row) pivoting, A row-major n x n overwritten, b overwritten with x.
 * Returns 0, or 1 if a zero / non-finite pivot column is met. */
int oracle_dense_solve(int n, double* A, double* b, int sp)
{
    int i, j, k;
    for (k = 0; k < n; ++k) {
        int p = k; double best = fabs(A[(size_t)k * n + k]);
        for (i = k + 1; i < n; ++i) { double v = fabs(A[(size_t)i * n + k]); if (v > best) { best = v; p = i; } }
        if (!(best > 0) || !isfinite(best)) return 1;
        if (p != k) {
            for (j = 0; j < n; ++j) { double tmp = A[(size_t)k * n + j]; A[(size_t)k * n + j] = A[(size_t)p * n + j]; A[(size_t)p * n + j] = tmp; }
            { double tmp = b[k]; b[k] = b[p]; b[p] = tmp; }
        }
        for (i = k + 1; i < n; ++i) {
            double l = A[(size_t)i * n + k];
            if (l == 0) continue;
            l = RND(sp, l / A[(size_t)k * n + k]);
            A[(size_t)i * n + k] = l;
            for (j = k + 1; j < n; ++j) {
                double u = A[(size_t)k * n + j];
                if (u != 0) A[(size_t)i * n + j] = RND(sp, A[(size_t)i * n + j] - RND(sp, l * u));
            }
            b[i] = RND(sp, b[i] - RND(sp, l * b[k]));
        }
    }
    for (k = n - 1; k >= 0; --k) {
        double s = b[k];
        for (j = k + 1; j < n; ++j) { double u = A[(size_t)k * n + j]; if (u != 0) s = RND(sp, s - RND(sp, u * b[j])); }
        b[k] = RND(sp, s / A[(size_t)k * n + k]);
    }
    return 0;
}

/* Textbook sparse Gaussian elimination with partial pivoting (right-looking, row storage).
 * Columns are eliminated in ascending order of their initial entry count (a static, deliberately
 * simple fill-reducing choice); in each column the pivot is the largest remaining entry.
 * A is given as COO (duplicates are summed).  b is overwritten with x.  Returns 0 / 1 (singular). */
typedef struct { int n, cap; int* c; double* v; } srow_t;
static void srow_push(srow_t* r, int c, double v) {
    if (r->n == r->cap) {
        r->cap = r->cap ? 2 * r->cap : 8;
        r->c = (int*)realloc(r->c, sizeof(int) * (size_t)r->cap);
        r->v = (double*)realloc(r->v, sizeof(double) * (size_t)r->cap);
    }
    r->c[r->n] = c; r->v[r->n] = v; r->n++;
}
typedef struct { int n, cap; int* r; } ilist_t;
static void ilist_push(ilist_t* l, int r) {
    if (l->n == l->cap) { l->cap = l->cap ? 2 * l->cap : 8; l->r = (int*)realloc(l->r, sizeof(int) * (size_t)l->cap); }
    l->r[l->n++] = r;
}
typedef struct { int key, idx; } keyidx_t;
static int keyidx_cmp(const void* a, const void* b) {
    const keyidx_t* x = (const keyidx_t*)a; const keyidx_t* y = (const keyidx_t*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);
}
int oracle_sparse_solve(int n, int nnz, const int* ar, const int* ac, const double* av, double* b, int sp)
{
    srow_t* row = (srow_t*)calloc((size_t)n, sizeof(srow_t));       /* active part of each row */
    ilist_t* cl = (ilist_t*)calloc((size_t)n, sizeof(ilist_t));     /* rows that ever held column c */
    int* pos = (int*)malloc(sizeof(int) * (size_t)n);               /* scratch: column -> slot in a row */
    int* done = (int*)calloc((size_t)n, sizeof(int));               /* row already used as a pivot row */
    int* prow = (int*)malloc(sizeof(int) * (size_t)n);              /* pivot row of step k */
    int* pcol = (int*)malloc(sizeof(int) * (size_t)n);              /* column eliminated at step k */
    double* x = (double*)malloc(sizeof(double) * (size_t)n);
    keyidx_t* ord = (keyidx_t*)malloc(sizeof(keyidx_t) * (size_t)n);
    int i, k, e, rc = 0;
    for (i = 0; i < n; ++i) { pos[i] = -1; ord[i].key = 0; ord[i].idx = i; }
    for (e = 0; e < nnz; ++e) {                                     /* load, summing duplicates */
        srow_t* r = &row[ar[e]]; int q, found = -1;
        for (q = 0; q < r->n; ++q) if (r->c[q] == ac[e]) { found = q; break; }
        if (found >= 0) r->v[found] += av[e];
        else { srow_push(r, ac[e], av[e]); ilist_push(&cl[ac[e]], ar[e]); ord[ac[e]].key++; }
    }
    if (sp) for (i = 0; i < n; ++i) { int q; for (q = 0; q < row[i].n; ++q) row[i].v[q] = (double)(float)row[i].v[q]; b[i] = (double)(float)b[i]; }
    qsort(ord, (size_t)n, sizeof(keyidx_t), keyidx_cmp);
    for (k = 0; k < n && !rc; ++k) {
        int c = ord[k].idx, p = -1, q; double best = 0, piv;
        ilist_t* L = &cl[c];
        for (q = 0; q < L->n; ++q) {                                /* choose the pivot row */
            int ri = L->r[q], s; if (done[ri]) continue;
            for (s = 0; s < row[ri].n; ++s) if (row[ri].c[s] == c) { double v = fabs(row[ri].v[s]); if (v > best) { best = v; p = ri; } break; }
        }
        if (p < 0 || !isfinite(best)) { rc = 1; break; }
        done[p] = 1; prow[k] = p; pcol[k] = c;
        piv = 0; for (q = 0; q < row[p].n; ++q) if (row[p].c[q] == c) piv = row[p].v[q];
        for (q = 0; q < L->n; ++q) {                                /* eliminate column c from the others */
            int ri = L->r[q], s, at = -1; double l; srow_t* R;
            if (done[ri]) continue;
            R = &row[ri];
            for (s = 0; s < R->n; ++s) if (R->c[s] == c) { at = s; break; }
            if (at < 0) continue;
            l = RND(sp, R->v[at] / piv);
            R->n--; R->c[at] = R->c[R->n]; R->v[at] = R->v[R->n];  /* drop (ri, c) */
            for (s = 0; s < R->n; ++s) pos[R->c[s]] = s;
            for (s = 0; s < row[p].n; ++s) {
                int j = row[p].c[s]; double u = row[p].v[s];
                if (j == c) continue;
                if (pos[j] >= 0) R->v[pos[j]] = RND(sp, R->v[pos[j]] - RND(sp, l * u));
                else { srow_push(R, j, RND(sp, -RND(sp, l * u))); pos[j] = R->n - 1; ilist_push(&cl[j], ri); }
            }
            for (s = 0; s < R->n; ++s) pos[R->c[s]] = -1;
            b[ri] = RND(sp, b[ri] - RND(sp, l * b[p]));
        }
    }
    if (!rc) {
        for (k = n - 1; k >= 0; --k) {                              /* back substitution */
            int p = prow[k], c = pcol[k], s; double sum = b[p], piv = 0;
            for (s = 0; s < row[p].n; ++s) {
                int j = row[p].c[s];
                if (j == c) piv = row[p].v[s]; else sum = RND(sp, sum - RND(sp, row[p].v[s] * x[j]));
            }
            x[c] = RND(sp, sum / piv);
        }
        memcpy(b, x, sizeof(double) * (size_t)n);
    }
    for (i = 0; i < n; ++i) { free(row[i].c); free(row[i].v); free(cl[i].r); }
    free(row); free(cl); free(pos); free(done); free(prow); free(pcol); free(x); free(ord);
    return rc;
}

/* solve A z = rhs with A in COO; method 0 = dense partial pivoting, 1 = sparse; transpose != 0 solves A^T. */
int oracle_linear_solve(int n, int nnz, const int* ar, const int* ac, const double* av, double* rhs,
                        int method, int transpose, int sp)
{
    const int* rr = transpose ? ac : ar; const int* cc = transpose ? ar : ac;
    if (method == 0) {
        double* A = (double*)calloc((size_t)n * (size_t)n, sizeof(double)); int e, rc;
        for (e = 0; e < nnz; ++e) A[(size_t)rr[e] * n + cc[e]] += av[e];
        if (sp) { size_t q; for (q = 0; q < (size_t)n * (size_t)n; ++q) A[q] = (double)(float)A[q]; for (e = 0; e < n; ++e) rhs[e] = (double)(float)rhs[e]; }
        rc = oracle_dense_solve(n, A, rhs, sp);
        free(A);
        return rc;
    }
    return oracle_sparse_solve(n, nnz, rr, cc, av, rhs, sp);
}

/* ----------------------------------------------------------------------------------------------- */
/* One scenario of Newton-Raphson (DESIGN.md loop convention):
 *   it = 0; loop { F, r = mismatch(V); if r <= tol: converged, stop; if it == max_it or r not finite:
 *   stop, not converged; solve J1 dz = -F; z += dz; ++it }
 * iterations = updates applied when converged, max_it otherwise.  norm_hist (may be NULL) receives r of
 * every evaluation, [max_it + 1] entries, NaN-padded. */
static void nr_one(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                   const uint8_t* bus_type, const int* th_idx, const int* vm_idx, int n,
                   const double* p_spec, const double* q_spec, const double* v_set,
                   const double* vm0, const double* va0, double tol, int max_it, int method, int mixed,
                   double* vm, double* va, int* iterations, uint8_t* converged, double* final_norm,
                   double* norm_hist)
{
    int nnzY = row_ptr[n_bus], cap = 4 * nnzY + 4 * n_bus, i, it = 0, conv = 0;
    double* F = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
    double* P = (double*)malloc(sizeof(double) * (size_t)n_bus);
    double* Q = (double*)malloc(sizeof(double) * (size_t)n_bus);
    int* jr = (int*)malloc(sizeof(int) * (size_t)cap);
    int* jc = (int*)malloc(sizeof(int) * (size_t)cap);
    double* jv = (double*)malloc(sizeof(double) * (size_t)cap);
    double r = 0;
    for (i = 0; i < n_bus; ++i) {      /* initial state: PAPER.md:287 flat start; PV / slack at setpoint */
        vm[i] = (bus_type[i] == PQ_BUS) ? (vm0 ? vm0[i] : 1.0) : v_set[i];
        va[i] = va0 ? va0[i] : 0.0;
    }
    if (norm_hist) for (i = 0; i <= max_it; ++i) norm_hist[i] = NAN;
    for (;;) {
        r = oracle_mismatch(n_bus, row_ptr, col, g, bb, bus_type, p_spec, q_spec, vm, va, th_idx, vm_idx, F, P, Q);
        if (norm_hist) norm_hist[it] = r;
        if (r <= tol) { conv = 1; break; }
        if (it == max_it || !isfinite(r)) break;
        {
            int m = oracle_jacobian_coo(n_bus, row_ptr, col, g, bb, vm, va, P, Q, th_idx, vm_idx, jr, jc, jv);
            for (i = 0; i < n; ++i) F[i] = -F[i];
            if (oracle_linear_solve(n, m, jr, jc, jv, F, method, 0, mixed)) { r = NAN; break; }
            for (i = 0; i < n_bus; ++i) {                           /* PAPER.md:90 update */
                if (th_idx[i] >= 0) va[i] += F[th_idx[i]];
                if (vm_idx[i] >= 0) vm[i] += F[vm_idx[i]];
            }
        }
        ++it;
    }
    *iterations = conv ? it : max_it;
    *converged = (uint8_t)conv;
    if (final_norm) *final_norm = r;
    free(F); free(P); free(Q); free(jr); free(jc); free(jv);
}

/* Batched NR: scenarios are independent (eq. 19) and are spread over host threads.
 * All per-scenario arrays are [batch][n_bus] row-major.  vm0/va0/final_norm/norm_hist may be NULL.
 * Returns the number of threads used. */
int oracle_nr_batch(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                    const uint8_t* bus_type, int batch, const double* p_spec, const double* q_spec,
                    const double* v_set, const double* vm0, const double* va0, double tol, int max_it,
                    int method, int mixed, int n_threads, double* vm, double* va, int* iterations,
                    uint8_t* converged, double* final_norm, double* norm_hist)
{
    int* th_idx = (int*)malloc(sizeof(int) * (size_t)n_bus);
    int* vm_idx = (int*)malloc(sizeof(int) * (size_t)n_bus);
    int n = oracle_index_maps(n_bus, bus_type, th_idx, vm_idx), s, used = 1;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
    used = n_threads < batch ? n_threads : (batch > 0 ? batch : 1);
#pragma omp parallel for schedule(dynamic, 1) num_threads(used)
#endif
    for (s = 0; s < batch; ++s) {
        size_t o = (size_t)s * (size_t)n_bus;
        nr_one(n_bus, row_ptr, col, g, bb, bus_type, th_idx, vm_idx, n, p_spec + o, q_spec + o, v_set + o,
               vm0 ? vm0 + o : NULL, va0 ? va0 + o : NULL, tol, max_it, method, mixed, vm + o, va + o,
               iterations + s, converged + s, final_norm ? final_norm + s : NULL,
               norm_hist ? norm_hist + (size_t)s * (size_t)(max_it + 1) : NULL);
    }
    free(th_idx); free(vm_idx);
    return used;
}

/* Batched adjoint, eq. (14): J1(V)^T lambda = g with J1 formed at the given (converged) V.
 * g_va[i] = dl/dtheta_i (slack ignored), g_vm[i] = dl/dVm_i (PQ only).  lam_p[i] multiplies the P_i
 * equation (0 at the slack), lam_q[i] the Q_i equation (0 off PQ).  With F = S_calc - S_spec,
 * lambda = d(g^T z1)/dS_spec.  Returns threads used. */
int oracle_adjoint_batch(int n_bus, const int* row_ptr, const int* col, const double* g, const double* bb,
                         const uint8_t* bus_type, int batch, const double* vm, const double* va,
                         const double* g_va, const double* g_vm, int method, int mixed, int n_threads,
                         double* lam_p, double* lam_q)
{
    int* th_idx = (int*)malloc(sizeof(int) * (size_t)n_bus);
    int* vm_idx = (int*)malloc(sizeof(int) * (size_t)n_bus);
    int n = oracle_index_maps(n_bus, bus_type, th_idx, vm_idx), s, used = 1;
    int cap = 4 * row_ptr[n_bus] + 4 * n_bus;
#ifdef _OPENMP
    if (n_threads <= 0) n_threads = omp_get_max_threads();
    used = n_threads < batch ? n_threads : (batch > 0 ? batch : 1);
#pragma omp parallel for schedule(dynamic, 1) num_threads(used)
#endif
    for (s = 0; s < batch; ++s) {
        size_t o = (size_t)s * (size_t)n_bus; int i, m;
        double* P = (double*)malloc(sizeof(double) * (size_t)n_bus);
        double* Q = (double*)malloc(sizeof(double) * (size_t)n_bus);
        double* rhs = (double*)malloc(sizeof(double) * (size_t)(n > 0 ? n : 1));
        int* jr = (int*)malloc(sizeof(int) * (size_t)cap);
        int* jc = (int*)malloc(sizeof(int) * (size_t)cap);
        double* jv = (double*)malloc(sizeof(double) * (size_t)cap);
        oracle_injections(n_bus, row_ptr, col, g, bb, vm + o, va + o, P, Q);
        m = oracle_jacobian_coo(n_bus, row_ptr, col, g, bb, vm + o, va + o, P, Q, th_idx, vm_idx, jr, jc, jv);
        for (i = 0; i < n_bus; ++i) {
            if (th_idx[i] >= 0) rhs[th_idx[i]] = g_va[o + i];
            if (vm_idx[i] >= 0) rhs[vm_idx[i]] = g_vm[o + i];
        }
        if (oracle_linear_solve(n, m, jr, jc, jv, rhs, method, 1, mixed)) for (i = 0; i < n; ++i) rhs[i] = NAN;
        for (i = 0; i < n_bus; ++i) {
            lam_p[o + i] = th_idx[i] >= 0 ? rhs[th_idx[i]] : 0.0;
            lam_q[o + i] = vm_idx[i] >= 0 ? rhs[vm_idx[i]] : 0.0;
        }
        free(P); free(Q); free(rhs); free(jr); free(jc); free(jv);
    }
    free(th_idx); free(vm_idx);
    return used;
}
