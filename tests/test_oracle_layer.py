"""Pins of the oracle's implicit-layer backward (NEXT row 2; eqs. 10-16): central finite differences of the
whole layer (re-solve Step 1 with the oracle's NR at tol 1e-13, recover Step 2 from the injections) -- no formula of
`oracle.layer_backward` is reused."""
import numpy as np
import pytest

import oracle
import sable_synth as S
from util import oracle_Y


def layer_forward(net, Y, p_gen, v_set, p_load, q_load):
    """y(x): solve Step 1, recover Step 2.  Returns the output buffer pieces (p_g, q_g, vm, va) as full-bus arrays."""
    ps = (p_gen - p_load)[None, :]
    qs = (-q_load)[None, :]
    res = oracle.nr_batch(Y, net.bus_type, ps, qs, v_set[None, :], tol=1e-13, max_it=40, method=0)
    assert res["converged"][0]
    vm, va = res["vm"][0], res["va"][0]
    P, Q = oracle.injections(Y, vm, va)
    return P + p_load, Q + q_load, vm, va


@pytest.mark.parametrize("cfg,seed", [(1, 3), (2, 4)])
def test_layer_backward_vs_finite_differences(cfg, seed):
    net = S.make_network(cfg)
    Y = oracle_Y(net)
    nb = net.n_bus
    rng = np.random.Generator(np.random.PCG64(seed))
    pv = net.bus_type == S.PV
    gen = net.bus_type != S.PQ
    w_pg, w_qg, w_vm, w_va = (rng.standard_normal(nb) for _ in range(4))
    w_pg[~gen] = 0; w_qg[~gen] = 0; w_va[net.bus_type == S.SLACK] = 0

    def loss(p_gen, v_set):
        pg, qg, vm, va = layer_forward(net, Y, p_gen, v_set, net.p_load, net.q_load)
        return w_pg @ pg + w_qg @ qg + w_vm @ vm + w_va @ va      # linear loss: dL/dy = the weights

    pg0, vs0 = net.p_gen.copy(), net.v_set.copy()
    _, _, vm, va = layer_forward(net, Y, pg0, vs0, net.p_load, net.q_load)
    # p_g at PV buses is an input: its direct partial is w_pg there; Vm at PV / slack likewise w_vm
    dx_pg, dx_vm = oracle.layer_backward(Y, net.bus_type, vm, va, w_pg, w_qg, w_vm, w_va)
    h = 1e-6
    idx_pv = np.flatnonzero(pv)[:6]
    for i in idx_pv:
        e = np.zeros(nb); e[i] = h
        fd = (loss(pg0 + e, vs0) - loss(pg0 - e, vs0)) / (2 * h)
        assert abs(fd - dx_pg[i]) <= 2e-6 * max(1.0, abs(fd)), (i, fd, dx_pg[i])
    for i in np.flatnonzero(gen)[:6]:
        e = np.zeros(nb); e[i] = h
        fd = (loss(pg0, vs0 + e) - loss(pg0, vs0 - e)) / (2 * h)
        assert abs(fd - dx_vm[i]) <= 2e-6 * max(1.0, abs(fd)), (i, fd, dx_vm[i])
    assert (dx_pg[~pv] == 0).all() and (dx_vm[~gen] == 0).all()


def test_layer_backward_reduces_to_adjoint_when_loss_sees_only_z1():
    """With dL/dz2 = 0 the chain (12)-(16) is lambda = J1^-T dL/dz1, dL/dp_g,PV = lambda_P: the oracle's own adjoint."""
    net = S.make_network(1)
    Y = oracle_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=1)
    res = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, tol=1e-12, max_it=30, method=0)
    gva, gvm = S.make_adjoint_rhs(net, batch=1)
    lp, lq, _ = oracle.adjoint_batch(Y, net.bus_type, res["vm"], res["va"], gva, gvm, method=0)
    z = np.zeros(net.n_bus)
    dx_pg, dx_vm = oracle.layer_backward(Y, net.bus_type, res["vm"][0], res["va"][0], z, z, gvm[0], gva[0])
    pv = net.bus_type == S.PV
    assert np.abs(dx_pg[pv] - lp[0][pv]).max() <= 1e-10 * max(1.0, np.abs(lp).max())


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_sparse_layer_backward_equals_dense(cfg):
    """The scipy.sparse restatement (used for configs 4-5, where the dense form does not fit) against the dense form."""
    net = S.make_network(cfg)
    Y = oracle_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=2)
    res = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, tol=1e-10, max_it=30, method=1)
    rng = np.random.Generator(np.random.PCG64(50 + cfg))
    for b in range(2):
        gl = [rng.standard_normal(net.n_bus) for _ in range(4)]
        d = oracle.layer_backward(Y, net.bus_type, res["vm"][b], res["va"][b], *gl)
        s = oracle.layer_backward_sparse(Y, net.bus_type, res["vm"][b], res["va"][b], *gl)
        sc = max(1.0, np.abs(d[0]).max(), np.abs(d[1]).max())
        assert np.abs(d[0] - s[0]).max() <= 1e-10 * sc and np.abs(d[1] - s[1]).max() <= 1e-10 * sc


def test_sparse_layer_backward_vs_finite_differences_cfg4():
    """Finite differences of the whole layer on the 2 000-bus config (a few input coordinates): pins the sparse form at
    a size where the dense one is not used."""
    net = S.make_network(4)
    Y = oracle_Y(net)
    nb = net.n_bus
    rng = np.random.Generator(np.random.PCG64(9))
    pv = net.bus_type == S.PV
    gen = net.bus_type != S.PQ
    w_pg, w_qg, w_vm, w_va = (rng.standard_normal(nb) for _ in range(4))
    w_pg[~gen] = 0; w_qg[~gen] = 0; w_va[net.bus_type == S.SLACK] = 0

    def loss(p_gen, v_set):
        pg, qg, vm, va = layer_forward(net, Y, p_gen, v_set, net.p_load, net.q_load)
        return w_pg @ pg + w_qg @ qg + w_vm @ vm + w_va @ va

    def layer_forward(net, Y, p_gen, v_set, p_load, q_load):
        res = oracle.nr_batch(Y, net.bus_type, (p_gen - p_load)[None, :], (-q_load)[None, :], v_set[None, :], tol=1e-12, max_it=40, method=1)
        assert res["converged"][0]
        vm, va = res["vm"][0], res["va"][0]
        P, Q = oracle.injections(Y, vm, va)
        return P + p_load, Q + q_load, vm, va

    pg0, vs0 = net.p_gen.copy(), net.v_set.copy()
    _, _, vm, va = layer_forward(net, Y, pg0, vs0, net.p_load, net.q_load)
    dx_pg, dx_vm = oracle.layer_backward_sparse(Y, net.bus_type, vm, va, w_pg, w_qg, w_vm, w_va)
    h = 1e-5
    for i in np.flatnonzero(pv)[[0, 7, 123]]:
        e = np.zeros(nb); e[i] = h
        fd = (loss(pg0 + e, vs0) - loss(pg0 - e, vs0)) / (2 * h)
        assert abs(fd - dx_pg[i]) <= 5e-5 * max(1.0, abs(fd), np.abs(dx_pg).max()), (i, fd, dx_pg[i])
    for i in np.flatnonzero(gen)[[0, 5, 200]]:
        e = np.zeros(nb); e[i] = h
        fd = (loss(pg0, vs0 + e) - loss(pg0, vs0 - e)) / (2 * h)
        assert abs(fd - dx_vm[i]) <= 5e-5 * max(1.0, abs(fd), np.abs(dx_vm).max()), (i, fd, dx_vm[i])
