// Host symbolic phase of the SABLE B200 library (run once per network; PAPER.md:185-197 delegates this to
// cuDSS "analysis", so nothing of it is prescribed by the paper -- see DESIGN.md "Symbolic phase").
//
// The template is BUS-LEVEL: every non-slack bus is one node carrying a 2x2 block of unknowns/equations
// (theta_i <-> P_i, Vm_i <-> Q_i).  A PV bus keeps its 2x2 slot with the Vm/Q half padded by the identity
// (row dVm = 0), so all blocks have one shape.  With that pairing the block pattern of J1 is the pattern of
// Y_bus without the slack row/column, it is structurally symmetric, and a symmetric permutation with
// block-diagonal pivots suffices (SURVEY.md §8(a) notes on a0).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace sable {

struct Template {
    int n_bus = 0, slack = -1, n_node = 0, n_pq = 0, n_pv = 0, n_level = 0;

    // nodes are numbered in elimination order, grouped by level; the slack has position n_node
    std::vector<int32_t> node_bus;      // [n_node]   bus index of node p
    std::vector<int32_t> bus_node;      // [n_bus]    node position of bus i (slack -> n_node)
    std::vector<uint8_t> node_pq;       // [n_node]   1 = PQ node (2 unknowns), 0 = PV node (theta only)
    std::vector<int32_t> node_level;    // [n_node]
    std::vector<int32_t> level_ptr;     // [n_level+1] nodes of level l are [level_ptr[l], level_ptr[l+1])

    // canonical Y_bus, rows of the non-slack buses in node order, columns as node positions (slack = n_node)
    std::vector<int32_t> yptr;          // [n_node+1]
    std::vector<int32_t> ycol;
    std::vector<double>  yg, yb;
    std::vector<int32_t> ydiag;         // [n_node] slot of Y(m,m)

    // canonical Y_bus of ALL buses in bus order (Step-2 recovery of the slack / PV injections)
    std::vector<int32_t> fptr, fcol;    // [n_bus+1], [nnz_y]
    std::vector<double>  fg, fb;

    // filled block pattern: pair p owned by node m couples m with a later node j:  {U(m,j), L(j,m)}
    std::vector<int32_t> pair_ptr;      // [n_node+1]
    std::vector<int32_t> pair_row;      // [n_pair] m
    std::vector<int32_t> pair_col;      // [n_pair] j
    std::vector<int32_t> pair_yu;       // [n_pair] slot of Y(m,j) in (ycol, yg, yb) or -1 for a fill pair
    std::vector<int32_t> pair_yl;       // [n_pair] slot of Y(j,m) or -1

    // numeric refactorisation as a static "pull" program:
    //   pair target p=(m,j):  U(m,j) = J(m,j) - sum_t L(m,k) U(k,j),  L(j,m) = (J(j,m) - sum_t L(j,k) U(k,m)) D_m^-1
    //                         with term_a[t] = pair (k,m) and term_b[t] = pair (k,j)
    //   diag target m:        D_m = J(m,m) - sum_t L(m,k) U(k,m) with dterm[t] = pair (k,m)
    std::vector<int32_t> term_ptr;      // [n_pair+1]
    std::vector<int32_t> term_a, term_b;
    std::vector<int32_t> dterm_ptr;     // [n_node+1]
    std::vector<int32_t> dterm;         // [n_pair] (every pair (k,m) appears once, in the list of m)

    // statistics (scalar counts refer to the unpadded pattern: a PV node contributes 1 row/column)
    int64_t nnz_y = 0, nnz_j = 0, nnz_lu = 0, n_pair_j = 0, lu_flops = 0;
    int32_t max_terms_pair = 0, max_terms_diag = 0, max_pairs_node = 0;
};

// Returns 0 on success; 1 = invalid argument, 2 = structural error (codes of sable_status).  `err` gets a message.
int build_template(int32_t n_bus, const int32_t* row_ptr, const int32_t* col_idx, const double* y_re,
                   const double* y_im, const uint8_t* bus_type, int32_t slack, Template& T, std::string& err);

}  // namespace sable
