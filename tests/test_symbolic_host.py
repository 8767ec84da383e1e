"""CPU-only tests of the host side of the library: the C ABI loads and exports what include/sable.h declares, and
the symbolic phase (sable_create with device = -1) produces a correct static program -- checked by running that
program in numpy on the ORACLE's Jacobian values and comparing with a dense solve.  No GPU compute here."""
import os
import re

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle
import sable_synth as S
from util import make_ctx, oracle_Y, random_state

import paper_2606_07099_b200 as sb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2606_07099_b200 import build
    build.build()


def test_library_exports_every_declared_symbol():
    hdr = open(os.path.join(ROOT, "include", "sable.h")).read()
    declared = set(re.findall(r"\b(sable_[a-z_0-9]+)\s*\(", hdr))
    assert {"sable_create", "sable_solve", "sable_adjoint", "sable_destroy"} <= declared
    L = sb.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in include/sable.h but not exported by libsable.so"
    assert declared == set(sb.EXPORTS)


def test_no_oracle_or_cpu_fallback_in_product():
    """The product path may not import the oracle (and the oracle may not import the product)."""
    for d, banned in (("paper_2606_07099_b200", "oracle"), ("oracle", "paper_2606_07099_b200")):
        for dirpath, _, files in os.walk(os.path.join(ROOT, d)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".c", ".h")):
                    txt = open(os.path.join(dirpath, f)).read()
                    assert not re.search(rf"^\s*(import|from)\s+{banned}\b", txt, re.M), (f, banned)
                    assert not re.search(rf"#include\s+\"[^\"]*{banned}", txt), (f, banned)
                    assert not re.search(rf"(CDLL|dlopen|import_module)\([^)]*{banned}", txt), (f, banned)


def closed_form_nnz_j(Y, bus_type):
    """SURVEY.md §8(a) notes: nnz(J1) = sum over stored Y_ij, i,j != slack, of (1+[i in PQ]) (1+[j in PQ])."""
    row_ptr, col, _, _ = Y
    w = np.where(bus_type == S.PQ, 2, np.where(bus_type == S.PV, 1, 0))
    tot = 0
    for i in range(len(bus_type)):
        tot += int(w[i] * w[col[row_ptr[i]:row_ptr[i + 1]]].sum())
    return tot


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_info_counts(cfg):
    net = S.make_network(cfg)
    Y = oracle_Y(net)
    ctx = make_ctx(net, max_batch=1, device=-1)
    I = ctx.info
    assert I["n_bus"] == net.n_bus and I["n_pv"] == net.cfg.n_pv and I["n_pq"] == net.n_bus - 1 - net.cfg.n_pv
    assert I["n"] == I["n_pv"] + 2 * I["n_pq"] == oracle.index_maps(net.bus_type)[0]
    assert I["nnz_y"] == net.n_bus + 2 * net.cfg.n_branch == len(Y[1])
    assert I["nnz_j"] == closed_form_nnz_j(Y, net.bus_type)
    assert I["nnz_lu"] >= I["nnz_j"] and I["n_node"] == net.n_bus - 1
    pat = ctx.debug_pattern()
    lvl = pat["node_level"]
    assert (np.diff(lvl) >= 0).all() and lvl[0] == 0 and lvl[-1] == I["n_level"] - 1
    assert sorted(pat["node_bus"].tolist()) == [i for i in range(net.n_bus) if i != net.slack]
    ctx.close()


def run_static_program(pat, Jblk_diag, Jblk_pair, rhs, transposed=False):
    """The device program of sable_stages.cuh, replayed in numpy FP64 from the exported lists (block 2x2)."""
    nn = len(pat["node_bus"])
    lvl = pat["node_level"]
    pp, pc = pat["pair_ptr"], pat["pair_col"]
    prow = np.repeat(np.arange(nn), np.diff(pp))
    dg = Jblk_diag.copy()
    U = Jblk_pair[:, 0].copy()
    L = Jblk_pair[:, 1].copy()
    y = rhs.copy()
    for l in range(lvl.max() + 1 if nn else 0):
        nodes = np.flatnonzero(lvl == l)
        for m in nodes:
            D = dg[m].copy()
            for q in range(pat["dterm_ptr"][m], pat["dterm_ptr"][m + 1]):
                a = pat["dterm"][q]
                assert pc[a] == m and lvl[prow[a]] < l
                D -= L[a] @ U[a]
                y[m] -= (U[a].T if transposed else L[a]) @ y[prow[a]]
            dg[m] = np.linalg.inv(D)
            if transposed:
                y[m] = dg[m].T @ y[m]
        for m in nodes:
            for p in range(pp[m], pp[m + 1]):
                for q in range(pat["term_ptr"][p], pat["term_ptr"][p + 1]):
                    a, b = pat["term_a"][q], pat["term_b"][q]
                    assert prow[a] == prow[b] and pc[a] == m and pc[b] == pc[p] and lvl[prow[a]] < l
                    U[p] -= L[a] @ U[b]
                    L[p] -= L[b] @ U[a]
                L[p] = L[p] @ dg[m]
    for l in range(lvl.max(), -1, -1):
        for m in np.flatnonzero(lvl == l):
            for p in range(pp[m], pp[m + 1]):
                assert lvl[pc[p]] > l
                y[m] -= (L[p].T if transposed else U[p]) @ y[pc[p]]
            if not transposed:
                y[m] = dg[m] @ y[m]
    return y


def blocks_from_oracle(net, Y, pat, vm, va):
    """The oracle's J1 laid out in the library's padded block layout; asserts every entry has a slot."""
    n, th, vmx = oracle.index_maps(net.bus_type)
    J = oracle.jacobian_dense(Y, net.bus_type, vm, va)
    _, jr, jc, _ = oracle.jacobian(Y, net.bus_type, vm, va)
    covered = np.zeros((n, n), bool)
    nb = pat["node_bus"]

    def blk(bi, bj):
        out = np.zeros((2, 2))
        rows, cols = (th[bi], vmx[bi]), (th[bj], vmx[bj])
        for a in range(2):
            for c in range(2):
                if rows[a] >= 0 and cols[c] >= 0:
                    out[a, c] = J[rows[a], cols[c]]
                    covered[rows[a], cols[c]] = True
                elif bi == bj and a == 1 and c == 1:
                    out[a, c] = 1.0
        return out

    nn = len(nb)
    diag = np.stack([blk(nb[m], nb[m]) for m in range(nn)]) if nn else np.zeros((0, 2, 2))
    prow = np.repeat(np.arange(nn), np.diff(pat["pair_ptr"]))
    pairs = np.zeros((len(prow), 2, 2, 2))
    for p, (m, j) in enumerate(zip(prow, pat["pair_col"])):
        pairs[p, 0] = blk(nb[m], nb[j])
        pairs[p, 1] = blk(nb[j], nb[m])
    assert covered[jr, jc].all(), "template misses a structural entry of J1"
    return J, diag, pairs, (n, th, vmx)


def check_program(net, seed, transposed):
    Y = oracle_Y(net)
    ctx = make_ctx(net, max_batch=1, device=-1)
    pat = ctx.debug_pattern()
    vm, va = random_state(net, 1, seed)
    J, diag, pairs, (n, th, vmx) = blocks_from_oracle(net, Y, pat, vm[0], va[0])
    rng = np.random.Generator(np.random.PCG64(seed))
    r = rng.standard_normal(n)
    nb = pat["node_bus"]
    rhs = np.zeros((len(nb), 2))
    for m, bus in enumerate(nb):
        rhs[m, 0] = r[th[bus]]
        if vmx[bus] >= 0:
            rhs[m, 1] = r[vmx[bus]]
    x = run_static_program(pat, diag, pairs, rhs, transposed)
    xr = np.linalg.solve(J.T if transposed else J, r)
    for m, bus in enumerate(nb):
        assert abs(x[m, 0] - xr[th[bus]]) <= 1e-9 * max(1, np.abs(xr).max())
        if vmx[bus] >= 0:
            assert abs(x[m, 1] - xr[vmx[bus]]) <= 1e-9 * max(1, np.abs(xr).max())
        else:
            assert x[m, 1] == 0.0
    ctx.close()


@pytest.mark.parametrize("cfg", [1, 2, 3])
@pytest.mark.parametrize("transposed", [False, True])
def test_static_program_solves_the_oracle_jacobian(cfg, transposed):
    check_program(S.make_network(cfg), 11 + cfg, transposed)


@settings(max_examples=25, deadline=None)
@given(n_bus=st.integers(2, 24), extra=st.integers(0, 6), pv_frac=st.floats(0, 1), seed=st.integers(1, 10_000),
       transposed=st.booleans())
def test_static_program_property(n_bus, extra, pv_frac, seed, transposed):
    extra = min(extra, max(0, (n_bus - 1) * (n_bus - 2) // 2 - 2)) if n_bus > 3 else 0
    n_pv = int(round(pv_frac * (n_bus - 1)))
    try:
        net = S.tiny_network(n_bus, extra, n_pv, seed)
    except RuntimeError:
        net = S.tiny_network(n_bus, 0, n_pv, seed)
    check_program(net, seed, transposed)


def test_fill_pattern_on_a_ring():
    """Hand-checkable: a ring of 6 buses (slack 0) leaves the path 1-2-3-4-5; minimum degree eliminates from the
    ends with no fill: 4 pairs, all in J1.  Adding the chord 1-5 closes the ring 1..5: one fill pair per
    elimination until three nodes remain: 5 ring pairs + 2 fill pairs."""
    def ring_ctx(chord):
        f = np.array([0, 1, 2, 3, 4, 5] + ([1] if chord else []), np.int32)
        t = np.array([1, 2, 3, 4, 5, 0] + ([5] if chord else []), np.int32)
        k = len(f)
        Y = S.ybus_triplets(6, f, t, np.full(k, 0.01), np.full(k, 0.1), np.zeros(k))
        return sb.Context(6, *Y, np.array([2, 0, 0, 0, 0, 0], np.uint8), 0, max_batch=1, device=-1)
    a, b = ring_ctx(False), ring_ctx(True)
    assert a.info["n_pair"] == 4 and a.info["n_pair_j"] == 4 and a.info["n_term"] == 0
    assert b.info["n_pair_j"] == 5 and b.info["n_pair"] == 7
    assert a.info["nnz_j"] == 4 * (5 + 2 * 4) and a.info["nnz_lu"] == a.info["nnz_j"]
    a.close(); b.close()


def test_create_rejects_bad_input():
    net = S.make_network(1)
    rp, ci, g, b = S.ybus_triplets(net.n_bus, net.f, net.t, net.r, net.x, net.b)
    bt = net.bus_type

    def status(*a, **k):
        with pytest.raises(sb.SableError) as e:
            sb.Context(*a, max_batch=1, device=-1, **k)
        return e.value.status
    bad = bt.copy(); bad[0] = 0
    assert status(net.n_bus, rp, ci, g, b, bad, 0) == 2                       # no slack
    bad = bt.copy(); bad[3] = 2
    assert status(net.n_bus, rp, ci, g, b, bad, 0) == 2                       # two slacks
    assert status(net.n_bus, rp, ci, g, b, bt, 1) == 2                        # slack index disagrees with bus_type
    ci2 = ci.copy(); ci2[5] = 99
    assert status(net.n_bus, rp, ci2, g, b, bt, 0) == 2                       # column out of range
    rp2 = rp.copy(); rp2[3] = rp2[2] - 1
    assert status(net.n_bus, rp2, ci, g, b, bt, 0) == 2                       # row_ptr not monotone
    assert status(1, rp[:2], ci, g, b, bt[:1], 0) == 1                        # n_bus < 2
    # an island: bus 13 cut off
    keep = (net.f != 13) & (net.t != 13)
    Y = S.ybus_triplets(net.n_bus, net.f[keep], net.t[keep], net.r[keep], net.x[keep], net.b[keep])
    assert status(net.n_bus, *Y, bt, 0) == 2
    with pytest.raises(sb.SableError) as e:
        sb.Context(net.n_bus, rp, ci, g, b, bt, 0, max_batch=0, device=-1)
    assert e.value.status == 1
    # host-only context: symbolic queries work, compute calls report STATE (no GPU is touched)
    ctx = sb.Context(net.n_bus, rp, ci, g, b, bt, 0, max_batch=2, device=-1)
    z = np.zeros((2, net.n_bus))
    with pytest.raises(sb.SableError) as e:
        ctx.solve_host(z, z, z + 1)
    assert e.value.status == 5
    ctx.close()


def test_create_canonicalises_unsorted_duplicate_input():
    """Unsorted columns, duplicate entries and a missing transpose entry give the same template as the clean CSR."""
    net = S.make_network(2)
    Yc = oracle_Y(net)                       # sorted, merged
    a = sb.Context(net.n_bus, *Yc, net.bus_type, 0, max_batch=1, device=-1)
    b = make_ctx(net, max_batch=1, device=-1)   # unsorted triplets with duplicates
    pa, pb = a.debug_pattern(), b.debug_pattern()
    for k in pa:
        assert np.array_equal(pa[k], pb[k]), k
    assert a.info == b.info
    a.close(); b.close()
