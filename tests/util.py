"""Shared helpers of the parity tests: build a network once, hand the SAME seeded arrays to the oracle
(oracle/) and to the CUDA library (paper_2606_07099_b200/), compare.  No arithmetic of the method here."""
from __future__ import annotations

import numpy as np

import oracle
import sable_synth as S


def oracle_Y(net):
    return oracle.ybus(net.n_bus, net.f, net.t, net.r, net.x, net.b)


def make_ctx(net, **opt):
    """sable_create on the harness-side Y_bus (unsorted triplets with duplicates: the library canonicalises)."""
    import paper_2606_07099_b200 as sb
    Y = S.ybus_triplets(net.n_bus, net.f, net.t, net.r, net.x, net.b)
    return sb.Context(net.n_bus, *Y, net.bus_type, net.slack, **opt)


def dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def random_state(net, batch, seed, spread=0.1):
    """A plausible non-flat state: |V| in [0.92, 1.08] at PQ buses, setpoints elsewhere, small angles."""
    rng = np.random.Generator(np.random.PCG64(seed))
    vm = np.repeat(net.v_set[None, :], batch, axis=0).copy()
    pq = net.bus_type == S.PQ
    vm[:, pq] = rng.uniform(0.92, 1.08, (batch, int(pq.sum())))
    va = rng.uniform(-spread, spread, (batch, net.n_bus))
    va[:, net.slack] = 0.0
    return vm, va


def gpu_jacobian_dense(ctx, net, diag, pairs):
    """Assemble the library's padded block layout (include/sable.h, sable_debug_jacobian) into the oracle's
    dense J1 ordering.  Returns (J [n][n], padding_ok)."""
    n, th, vmx = oracle.index_maps(net.bus_type)
    pat = ctx.debug_pattern()
    nb = pat["node_bus"]
    J = np.zeros((n, n))
    seen = np.zeros((n, n), dtype=bool)
    pad_ok = True

    def put(bi, bj, blk):
        nonlocal pad_ok
        rows = (th[bi], vmx[bi])
        cols = (th[bj], vmx[bj])
        for a in range(2):
            for c in range(2):
                v = blk[2 * a + c]
                if rows[a] >= 0 and cols[c] >= 0:
                    J[rows[a], cols[c]] = v
                    seen[rows[a], cols[c]] = True
                else:   # padded slot of a PV node: 0 off the diagonal, 1 at dQ/dVm of the node itself
                    want = 1.0 if (bi == bj and a == 1 and c == 1) else 0.0
                    pad_ok = pad_ok and (v == want)

    for m in range(len(nb)):
        put(nb[m], nb[m], diag[m])
        for p in range(pat["pair_ptr"][m], pat["pair_ptr"][m + 1]):
            j = pat["pair_col"][p]
            put(nb[m], nb[j], pairs[p][0:4])
            put(nb[j], nb[m], pairs[p][4:8])
    return J, seen, pad_ok


def gpu_jacobian_coo(ctx, net, diag, pairs):
    """The library's padded block layout as COO triplets in the oracle's J1 ordering (for grids where the dense form
    does not fit).  Returns (rows, cols, vals, padding_ok)."""
    n, th, vmx = oracle.index_maps(net.bus_type)
    pat = ctx.debug_pattern()
    nb = pat["node_bus"].astype(np.int64)
    nn = nb.shape[0]
    prow = np.repeat(np.arange(nn), np.diff(pat["pair_ptr"]))
    pcol = pat["pair_col"].astype(np.int64)
    bi = np.concatenate([nb, nb[prow], nb[pcol]])
    bj = np.concatenate([nb, nb[pcol], nb[prow]])
    blk = np.concatenate([diag.reshape(nn, 4), pairs[:, 0:4], pairs[:, 4:8]])
    is_diag = np.concatenate([np.ones(nn, bool), np.zeros(2 * prow.shape[0], bool)])
    rows, cols, vals = [], [], []
    pad_ok = True
    for a, rmap in enumerate((th, vmx)):
        for c, cmap in enumerate((th, vmx)):
            r, cc, v = rmap[bi], cmap[bj], blk[:, 2 * a + c]
            real = (r >= 0) & (cc >= 0)
            rows.append(r[real]); cols.append(cc[real]); vals.append(v[real])
            want = np.where(is_diag & (a == 1) & (c == 1), 1.0, 0.0)
            pad_ok = pad_ok and bool((v[~real] == want[~real]).all())
    return np.concatenate(rows), np.concatenate(cols), np.concatenate(vals), pad_ok
