"""Pins for the CPU oracle (oracle/): everything here checks the oracle against something other than
itself -- closed forms, a hand-derived worked example, finite differences, complex-matrix identities
written with numpy, branch-flow power balance, numpy / scipy linear solves, and invariants.
Citations are PAPER.md lines (the method) and SURVEY.md §8(c) (the pins)."""
import json
import os

import numpy as np
import pytest
import scipy.sparse as sp
import scipy.sparse.linalg as spla

import oracle
import sable_synth as S


# ---------------------------------------------------------------------------------------------------
# helpers that deliberately do NOT reuse the oracle's formulas
def ybus_dense_numpy(net):
    """Y_bus as a dense complex matrix straight from the pi-model definition."""
    Y = np.zeros((net.n_bus, net.n_bus), dtype=complex)
    for f, t, r, x, b in zip(net.f, net.t, net.r, net.x, net.b):
        y = 1.0 / complex(r, x)
        Y[f, f] += y + 0.5j * b
        Y[t, t] += y + 0.5j * b
        Y[f, t] -= y
        Y[t, f] -= y
    return Y


def complex_injection(Yd, vm, va):
    """S = V o conj(Y V) (BASELINE.json north_star)."""
    V = vm * np.exp(1j * va)
    return V * np.conj(Yd @ V)


def random_state(net, rng, spread=0.15):
    vm = rng.uniform(0.92, 1.08, net.n_bus)
    va = rng.uniform(-spread, spread, net.n_bus)
    va[net.slack] = 0.0
    return vm, va


def csr_to_dense(Y, n):
    row_ptr, col, g, b = Y
    D = np.zeros((n, n), dtype=complex)
    for i in range(n):
        for k in range(row_ptr[i], row_ptr[i + 1]):
            D[i, col[k]] += complex(g[k], b[k])
    return D


def net_Y(net):
    return oracle.ybus(net.n_bus, net.f, net.t, net.r, net.x, net.b)


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("E,r,x,P,Q", [(1.03, 0.02, 0.09, 0.8, 0.3), (1.0, 0.01, 0.05, 0.5, 0.1),
                                       (1.05, 0.03, 0.10, 1.2, 0.4), (0.98, 0.0, 0.2, 0.3, -0.1)])
def test_two_bus_closed_form(E, r, x, P, Q):
    """slack E<0, one PQ bus with load P+jQ behind r+jx, no charging:
    v = |V2|^2 = 1/2 [E^2 - 2(rP+xQ) + sqrt((E^2 - 2(rP+xQ))^2 - 4 (r^2+x^2)(P^2+Q^2))],
    theta2 = -atan2(xP - rQ, v + rP + xQ)."""
    Y = oracle.ybus(2, [0], [1], [r], [x], [0.0])
    res = oracle.nr_batch(Y, [2, 0], np.array([[0.0, -P]]), np.array([[0.0, -Q]]), np.array([[E, 1.0]]),
                          tol=1e-13, max_it=20, method=0)
    a = E * E - 2 * (r * P + x * Q)
    v = 0.5 * (a + np.sqrt(a * a - 4 * (r * r + x * x) * (P * P + Q * Q)))
    assert res["converged"][0] == 1
    assert abs(res["vm"][0, 1] - np.sqrt(v)) < 1e-13
    assert abs(res["va"][0, 1] - (-np.arctan2(x * P - r * Q, v + r * P + x * Q))) < 1e-13
    assert res["vm"][0, 0] == E and res["va"][0, 0] == 0.0


def test_two_bus_survey_numbers():
    """Worked numbers quoted in SURVEY.md §8(c) for (E=1.03, r=0.02, x=0.09, P=0.8, Q=0.3)."""
    Y = oracle.ybus(2, [0], [1], [0.02], [0.09], [0.0])
    res = oracle.nr_batch(Y, [2, 0], np.array([[0.0, -0.8]]), np.array([[0.0, -0.3]]), np.array([[1.03, 1.0]]),
                          tol=1e-14, max_it=20, method=1)
    assert abs(res["vm"][0, 1] - 0.984120490568773) < 5e-15
    assert abs(res["va"][0, 1] + 0.065157705342144) < 5e-15
    assert res["iterations"][0] == 4


def test_three_bus_worked_example(golden_dir):
    gd = json.load(open(os.path.join(golden_dir, "three_bus_survey.json")))
    br = np.array(gd["branches_f_t_r_x_b"])
    Y = oracle.ybus(3, br[:, 0].astype(int), br[:, 1].astype(int), br[:, 2], br[:, 3], br[:, 4])
    Yd = csr_to_dense(Y, 3)
    assert abs(Yd[1, 1] - complex(gd["G11"], gd["B11"])) < 1e-13
    assert abs(Yd[1, 2] - complex(gd["G12"], gd["B12"])) < 1e-13
    assert abs(Yd[2, 2].imag - gd["B22"]) < 1e-13
    bt = gd["bus_type"]
    vs, ps, qs = np.array([gd["v_set"]]), np.array([gd["p_spec"]]), np.array([gd["q_spec"]])
    F, r0, _, _ = oracle.mismatch(Y, bt, ps[0], qs[0], [1.05, 1.02, 1.0], [0, 0, 0])
    np.testing.assert_allclose(F, gd["F_flat"], atol=1e-14)          # oracle order = [P1, P2, Q2]
    J = oracle.jacobian_dense(Y, bt, [1.05, 1.02, 1.0], [0, 0, 0])    # columns [th1, th2, vm2]
    np.testing.assert_allclose(J, gd["J_flat_rows_P1_P2_Q2_cols_th1_th2_vm2"], atol=1e-13)
    n, jr, jc, jv = oracle.jacobian(Y, bt, [1.05, 1.02, 1.0], [0, 0, 0])
    for method in (0, 1):
        dz = oracle.linear_solve(n, jr, jc, jv, -F, method=method)
        np.testing.assert_allclose(dz, gd["dz_first"], atol=2e-15)
    for method in (0, 1):
        res = oracle.nr_batch(Y, bt, ps, qs, vs, tol=1e-8, max_it=20, method=method, want_hist=True)
        assert res["iterations"][0] == gd["iterations"] and res["converged"][0] == 1
        np.testing.assert_allclose(res["hist"][0, :4], gd["norm_hist"], rtol=2e-6)
        assert abs(res["vm"][0, 2] - gd["vm2"]) < 1e-10
        assert abs(res["va"][0, 1] - gd["th1"]) < 1e-10 and abs(res["va"][0, 2] - gd["th2"]) < 1e-10
        Sc = complex_injection(Yd, res["vm"][0], res["va"][0])
        assert abs(Sc[0] - complex(*gd["slack_injection"])) < 1e-9
        assert abs(Sc[1].imag - gd["pv_q_injection"]) < 1e-9
        assert abs(Sc.sum() - complex(*gd["losses"])) < 1e-9
        g = gd["adjoint_g_th1_th2_vm2"]
        lp, lq, _ = oracle.adjoint_batch(Y, bt, res["vm"], res["va"], np.array([[0.0, g[0], g[1]]]),
                                         np.array([[0.0, 0.0, g[2]]]), method=method)
        np.testing.assert_allclose([lp[0, 1], lp[0, 2], lq[0, 2]], gd["adjoint_lambda_P1_P2_Q2"], atol=1e-9)
        assert lp[0, 0] == 0 and lq[0, 0] == 0 and lq[0, 1] == 0


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2])
def test_ybus_against_definition(cfg):
    net = S.make_network(cfg)
    Y = net_Y(net)
    row_ptr, col, g, b = Y
    Yd = ybus_dense_numpy(net)
    np.testing.assert_allclose(csr_to_dense(Y, net.n_bus), Yd, atol=1e-12)
    assert row_ptr[-1] == net.n_bus + 2 * net.f.shape[0]              # no parallel branches
    for i in range(net.n_bus):                                        # sorted, unique, diagonal present
        c = col[row_ptr[i]:row_ptr[i + 1]]
        assert np.all(np.diff(c) > 0) and i in c
    # row sums of Y are the shunt (charging) terms only
    shunt = np.zeros(net.n_bus)
    np.add.at(shunt, net.f, 0.5 * net.b)
    np.add.at(shunt, net.t, 0.5 * net.b)
    np.testing.assert_allclose(Yd.sum(axis=1), 1j * shunt, atol=1e-9)


@pytest.mark.parametrize("cfg", [1, 2])
def test_injections_complex_form_and_power_balance(cfg):
    """Real form of PAPER.md:201-207 against S = V conj(YV), and sum_i S_i = sum of branch losses
    S_ft + S_tf with S_ft = V_f conj((y + jb/2) V_f - y V_t) for ANY V."""
    net = S.make_network(cfg)
    Y = net_Y(net)
    Yd = ybus_dense_numpy(net)
    rng = np.random.default_rng(5)
    for _ in range(3):
        vm, va = random_state(net, rng)
        P, Q = oracle.injections(Y, vm, va)
        Sc = complex_injection(Yd, vm, va)
        np.testing.assert_allclose(P + 1j * Q, Sc, atol=1e-12)
        V = vm * np.exp(1j * va)
        loss = 0
        for f, t, r, x, b in zip(net.f, net.t, net.r, net.x, net.b):
            y = 1.0 / complex(r, x)
            loss += V[f] * np.conj((y + 0.5j * b) * V[f] - y * V[t]) + V[t] * np.conj((y + 0.5j * b) * V[t] - y * V[f])
        assert abs((P + 1j * Q).sum() - loss) < 1e-10


def test_mismatch_rows_sign_and_norm():
    net = S.make_network(1)
    Y = net_Y(net)
    Yd = ybus_dense_numpy(net)
    ps, qs, vs = S.make_scenarios(net, batch=1)
    rng = np.random.default_rng(1)
    vm, va = random_state(net, rng)
    F, r, P, Q = oracle.mismatch(Y, net.bus_type, ps[0], qs[0], vm, va)
    Sc = complex_injection(Yd, vm, va)
    nonslack = np.flatnonzero(net.bus_type != S.SLACK)
    pq = np.flatnonzero(net.bus_type == S.PQ)
    expect = np.concatenate([Sc.real[nonslack] - ps[0][nonslack], Sc.imag[pq] - qs[0][pq]])   # F = S_calc - S_spec
    np.testing.assert_allclose(F, expect, atol=1e-12)
    assert F.shape[0] == net.cfg.n_pv + 2 * pq.shape[0]                # n = n_PV + 2 n_PQ
    assert r == np.abs(F).max()


@pytest.mark.parametrize("cfg", [1, 2])
def test_jacobian_vs_finite_differences(cfg):
    """north_star: analytic Jacobian versus central finite differences, relative error <= 1e-6."""
    net = S.make_network(cfg)
    Y = net_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=1)
    rng = np.random.default_rng(11)
    vm, va = random_state(net, rng)
    n, th, vmx = oracle.index_maps(net.bus_type)
    J = oracle.jacobian_dense(Y, net.bus_type, vm, va)
    h = 1e-6
    Jfd = np.zeros_like(J)
    for i in range(net.n_bus):
        for idx, which in ((th[i], "a"), (vmx[i], "m")):
            if idx < 0:
                continue
            vp, ap, vn, an = vm.copy(), va.copy(), vm.copy(), va.copy()
            if which == "a":
                ap[i] += h; an[i] -= h
            else:
                vp[i] += h; vn[i] -= h
            Fp = oracle.mismatch(Y, net.bus_type, ps[0], qs[0], vp, ap)[0]
            Fn = oracle.mismatch(Y, net.bus_type, ps[0], qs[0], vn, an)[0]
            Jfd[:, idx] = (Fp - Fn) / (2 * h)
    assert np.abs(J - Jfd).max() <= 1e-6 * np.abs(J).max()
    # structural zeros of the FD Jacobian are zeros of the analytic one
    assert np.all(np.abs(J[np.abs(Jfd) < 1e-9]) < 1e-9)


@pytest.mark.parametrize("cfg", [1, 2])
def test_jacobian_vs_complex_identities(cfg):
    """dS/dtheta = j diag(V) conj(diag(I) - Y diag(V));  dS/dVm = diag(V) conj(Y diag(V/|V|)) +
    conj(diag(I)) diag(V/|V|)  (second independent form)."""
    net = S.make_network(cfg)
    Y = net_Y(net)
    Yd = ybus_dense_numpy(net)
    rng = np.random.default_rng(3)
    vm, va = random_state(net, rng)
    V = vm * np.exp(1j * va)
    I = Yd @ V
    dS_dth = 1j * np.diag(V) @ np.conj(np.diag(I) - Yd @ np.diag(V))
    dS_dvm = np.diag(V) @ np.conj(Yd @ np.diag(V / vm)) + np.conj(np.diag(I)) @ np.diag(V / vm)
    nonslack = np.flatnonzero(net.bus_type != S.SLACK)
    pq = np.flatnonzero(net.bus_type == S.PQ)
    Jc = np.block([[dS_dth.real[np.ix_(nonslack, nonslack)], dS_dvm.real[np.ix_(nonslack, pq)]],
                   [dS_dth.imag[np.ix_(pq, nonslack)], dS_dvm.imag[np.ix_(pq, pq)]]])
    J = oracle.jacobian_dense(Y, net.bus_type, vm, va)
    np.testing.assert_allclose(J, Jc, atol=1e-11 * np.abs(Jc).max())


def test_jacobian_pattern_count():
    """nnz(J1) = sum over stored Y_ij, i,j != slack, of (1+[i in PQ])(1+[j in PQ]) (SURVEY.md §8(a) notes)."""
    for cfg in (1, 2, 3):
        net = S.make_network(cfg)
        Y = net_Y(net)
        row_ptr, col, _, _ = Y
        n, jr, jc, jv = oracle.jacobian(Y, net.bus_type, np.ones(net.n_bus), np.zeros(net.n_bus))
        w = np.where(net.bus_type == S.PQ, 2, np.where(net.bus_type == S.PV, 1, 0))
        expect = sum(int(w[i]) * int(w[col[k]]) for i in range(net.n_bus) for k in range(row_ptr[i], row_ptr[i + 1]))
        assert jv.shape[0] == expect
        assert len(set(zip(jr.tolist(), jc.tolist()))) == expect       # no duplicates


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_linear_solvers_against_numpy_and_scipy(cfg):
    net = S.make_network(cfg)
    Y = net_Y(net)
    rng = np.random.default_rng(7)
    vm, va = random_state(net, rng)
    n, jr, jc, jv = oracle.jacobian(Y, net.bus_type, vm, va)
    A = sp.coo_matrix((jv, (jr, jc)), shape=(n, n)).tocsc()
    rhs = rng.standard_normal(n)
    x_np = np.linalg.solve(A.toarray(), rhs)
    x_sp = spla.splu(A).solve(rhs)
    scale = np.abs(x_np).max()
    for method in (0, 1):
        x = oracle.linear_solve(n, jr, jc, jv, rhs, method=method)
        assert np.abs(x - x_np).max() <= 1e-10 * scale
        assert np.abs(x - x_sp).max() <= 1e-10 * scale
        assert np.abs(A @ x - rhs).max() <= 1e-12 * max(1.0, np.abs(A).max() * scale)
        xt = oracle.linear_solve(n, jr, jc, jv, rhs, method=method, transpose=True)
        assert np.abs(xt - np.linalg.solve(A.toarray().T, rhs)).max() <= 1e-10 * np.abs(xt).max()


@pytest.mark.parametrize("cfg", [4, 5])
def test_sparse_solver_against_scipy_at_large_sizes(cfg):
    """Configs 4-5 (n = 3 598 / 17 036): the sparse elimination is the only oracle path used there, so it is cross-checked
    against scipy's SuperLU (plain and transposed) and by the residual at exactly those sizes."""
    net = S.make_network(cfg)
    Y = net_Y(net)
    rng = np.random.default_rng(11 + cfg)
    vm, va = random_state(net, rng)
    n, jr, jc, jv = oracle.jacobian(Y, net.bus_type, vm, va)
    A = sp.coo_matrix((jv, (jr, jc)), shape=(n, n)).tocsc()
    rhs = rng.standard_normal(n)
    lu = spla.splu(A)
    for transpose in (False, True):
        x_sp = lu.solve(rhs, trans="T" if transpose else "N")
        x = oracle.linear_solve(n, jr, jc, jv, rhs, method=1, transpose=transpose)
        scale = np.abs(x_sp).max()
        assert np.abs(x - x_sp).max() <= 1e-9 * scale
        M = A.T if transpose else A
        assert np.abs(M @ x - rhs).max() <= 1e-11 * max(1.0, np.abs(A).max() * scale)


def test_sparse_solver_pivots_when_needed():
    """A matrix whose natural diagonal is zero needs row exchanges; duplicates in COO are summed."""
    A = np.array([[0.0, 2.0, 0.0, 1.0], [1.0, 0.0, 3.0, 0.0], [0.0, 1e-9, 0.0, 4.0], [2.0, 0.0, 1.0, 0.0]])
    r, c = np.nonzero(A)
    v = A[r, c]
    r2, c2, v2 = np.concatenate([r, [0]]), np.concatenate([c, [1]]), np.concatenate([v, [0.5]])
    A2 = A.copy(); A2[0, 1] += 0.5
    b = np.array([1.0, -2.0, 0.5, 3.0])
    for method in (0, 1):
        np.testing.assert_allclose(oracle.linear_solve(4, r2, c2, v2, b, method=method), np.linalg.solve(A2, b), rtol=1e-12)
    with pytest.raises(np.linalg.LinAlgError):
        oracle.linear_solve(2, [0, 1], [0, 0], [1.0, 1.0], [1.0, 1.0], method=1)
    with pytest.raises(np.linalg.LinAlgError):
        oracle.linear_solve(2, [0, 1], [0, 0], [1.0, 1.0], [1.0, 1.0], method=0)


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,batch", [(1, 8), (2, 6), (3, 4)])
def test_nr_solution_properties(cfg, batch):
    net = S.make_network(cfg)
    Y = net_Y(net)
    Yd = ybus_dense_numpy(net)
    ps, qs, vs = S.make_scenarios(net, batch=batch)
    res0 = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, tol=1e-8, max_it=net.cfg.max_it, method=0, want_hist=True)
    res1 = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, tol=1e-8, max_it=net.cfg.max_it, method=1, want_hist=True)
    assert res0["converged"].all() and res1["converged"].all()
    np.testing.assert_array_equal(res0["iterations"], res1["iterations"])
    np.testing.assert_allclose(res0["vm"], res1["vm"], atol=1e-11)
    np.testing.assert_allclose(res0["va"], res1["va"], atol=1e-11)
    nonslack = net.bus_type != S.SLACK
    pq = net.bus_type == S.PQ
    for s in range(batch):
        Sc = complex_injection(Yd, res1["vm"][s], res1["va"][s])
        assert np.abs(Sc.real[nonslack] - ps[s][nonslack]).max() <= 1e-8      # the PF equations hold
        assert np.abs(Sc.imag[pq] - qs[s][pq]).max() <= 1e-8
        np.testing.assert_array_equal(res1["vm"][s][~pq], vs[s][~pq])         # PV / slack stay at setpoints
        assert res1["va"][s][net.slack] == 0.0
        h = res1["hist"][s]
        it = res1["iterations"][s]
        assert h[it] <= 1e-8 and (it == 0 or h[it - 1] > 1e-8) and np.all(np.isnan(h[it + 1:]))
        if it >= 3:                                                            # quadratic contraction at the end
            assert h[it - 1] <= 50 * h[it - 2] ** 2 + 1e-12
        # power balance with recovered slack / PV injections (north_star: to 1e-10 p.u. vs branch losses)
        V = res1["vm"][s] * np.exp(1j * res1["va"][s])
        loss = sum(V[f] * np.conj((1 / complex(r, x) + 0.5j * b) * V[f] - V[t] / complex(r, x)) +
                   V[t] * np.conj((1 / complex(r, x) + 0.5j * b) * V[t] - V[f] / complex(r, x))
                   for f, t, r, x, b in zip(net.f, net.t, net.r, net.x, net.b))
        assert abs(Sc.sum() - loss) <= 1e-10


def test_nr_invariances():
    net = S.make_network(2)
    Y = net_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=6)
    base = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=1)
    # batch order / composition / thread count
    perm = np.array([3, 0, 5, 1, 4, 2])
    shuf = oracle.nr_batch(Y, net.bus_type, ps[perm], qs[perm], vs[perm], method=1, n_threads=1)
    np.testing.assert_array_equal(shuf["vm"], base["vm"][perm])
    np.testing.assert_array_equal(shuf["iterations"], base["iterations"][perm])
    one = oracle.nr_batch(Y, net.bus_type, ps[2:3], qs[2:3], vs[2:3], method=1)
    np.testing.assert_array_equal(one["vm"][0], base["vm"][2])
    same = oracle.nr_batch(Y, net.bus_type, np.repeat(ps[:1], 4, 0), np.repeat(qs[:1], 4, 0), np.repeat(vs[:1], 4, 0), method=1)
    assert np.all(same["vm"] == same["vm"][0]) and np.all(same["va"] == same["va"][0])
    # bus relabelling
    rng = np.random.default_rng(0)
    p = rng.permutation(net.n_bus)            # new label of old bus i is p[i]
    inv = np.argsort(p)
    Yp = oracle.ybus(net.n_bus, p[net.f], p[net.t], net.r, net.x, net.b)
    rel = oracle.nr_batch(Yp, net.bus_type[inv], ps[:, inv], qs[:, inv], vs[:, inv], method=1)
    np.testing.assert_array_equal(rel["iterations"], base["iterations"])
    np.testing.assert_allclose(rel["vm"][:, p], base["vm"], atol=1e-10)
    np.testing.assert_allclose(rel["va"][:, p], base["va"], atol=1e-10)


def test_nr_conventions_and_edge_cases():
    net = S.make_network(2)
    Y = net_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=3)
    full = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=1)
    # iteration cap: not an error, converged = 0, iterations = max_it (reading 18)
    cap = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, max_it=2, method=1)
    assert not cap["converged"].any() and np.all(cap["iterations"] == 2) and np.all(cap["final_norm"] > 1e-8)
    # warm start at the solution: zero iterations
    warm = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, vm0=full["vm"], va0=full["va"], method=1)
    assert warm["converged"].all() and np.all(warm["iterations"] == 0)
    np.testing.assert_array_equal(warm["vm"], full["vm"])
    # non-finite input: frozen, not converged, iterations = max_it
    bad = ps.copy(); bad[1, 5] = np.nan
    nanr = oracle.nr_batch(Y, net.bus_type, bad, qs, vs, method=1)
    assert nanr["converged"].tolist() == [1, 0, 1] and nanr["iterations"][1] == 20
    np.testing.assert_array_equal(nanr["vm"][[0, 2]], full["vm"][[0, 2]])
    # infeasible load: diverges or stalls, flagged, never crashes
    heavy = oracle.nr_batch(Y, net.bus_type, ps * 40, qs * 40, vs, method=1)
    assert not heavy["converged"].any() and np.all(heavy["iterations"] == 20)


@pytest.mark.parametrize("n_pv", [0, 9])
def test_all_pq_and_all_pv_networks(n_pv):
    net = S.tiny_network(10, 4, n_pv, seed=3)
    Y = net_Y(net)
    Yd = ybus_dense_numpy(net)
    ps, qs, vs = S.make_scenarios(net, batch=4)
    if n_pv == 9:                                     # all PV: give the PV buses some injections to carry
        ps = ps + np.random.default_rng(1).uniform(-0.3, 0.3, ps.shape) * (net.bus_type == S.PV)
    for method in (0, 1):
        res = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=method)
        assert res["converged"].all()
        for s in range(4):
            Sc = complex_injection(Yd, res["vm"][s], res["va"][s])
            assert np.abs(Sc.real[1:] - ps[s][1:]).max() <= 1e-8
    n, _, _ = oracle.index_maps(net.bus_type)
    assert n == (18 if n_pv == 0 else 9)


# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg", [1, 2])
def test_adjoint_vs_finite_difference_sensitivities(cfg):
    """lambda_k = d(g^T z1)/dS_spec,k by central differences of full re-solves (tol 1e-13, h = 1e-6)."""
    net = S.make_network(cfg)
    Y = net_Y(net)
    ps, qs, vs = S.make_scenarios(net, batch=1)
    gva, gvm = S.make_adjoint_rhs(net, batch=1)
    sol = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, tol=1e-13, max_it=30, method=0)
    assert sol["converged"][0]
    lp, lq, _ = oracle.adjoint_batch(Y, net.bus_type, sol["vm"], sol["va"], gva, gvm, method=0)
    lp1, lq1, _ = oracle.adjoint_batch(Y, net.bus_type, sol["vm"], sol["va"], gva, gvm, method=1)
    np.testing.assert_allclose(lp1, lp, atol=1e-10 * np.abs(lp).max())
    np.testing.assert_allclose(lq1, lq, atol=1e-10 * np.abs(lp).max())
    assert lp[0, net.slack] == 0 and np.all(lq[0, net.bus_type != S.PQ] == 0)

    def obj(p, q):
        r = oracle.nr_batch(Y, net.bus_type, p, q, vs, tol=1e-13, max_it=30, method=0)
        return float((gva * r["va"]).sum() + (gvm * r["vm"]).sum())
    h = 1e-6
    rng = np.random.default_rng(2)
    nonslack = np.flatnonzero(net.bus_type != S.SLACK)
    pq = np.flatnonzero(net.bus_type == S.PQ)
    scale = max(np.abs(lp).max(), np.abs(lq).max())
    for k in rng.choice(nonslack, size=min(6, nonslack.shape[0]), replace=False):
        pp, pn = ps.copy(), ps.copy(); pp[0, k] += h; pn[0, k] -= h
        fd = (obj(pp, qs) - obj(pn, qs)) / (2 * h)
        assert abs(fd - lp[0, k]) <= 1e-6 * scale
    for k in rng.choice(pq, size=min(6, pq.shape[0]), replace=False):
        qp, qn = qs.copy(), qs.copy(); qp[0, k] += h; qn[0, k] -= h
        fd = (obj(ps, qp) - obj(ps, qn)) / (2 * h)
        assert abs(fd - lq[0, k]) <= 1e-6 * scale


def test_adjoint_is_transposed_solve():
    net = S.make_network(1)
    Y = net_Y(net)
    rng = np.random.default_rng(4)
    vm, va = random_state(net, rng)
    gva, gvm = S.make_adjoint_rhs(net, batch=1)
    n, th, vmx = oracle.index_maps(net.bus_type)
    J = oracle.jacobian_dense(Y, net.bus_type, vm, va)
    g = np.zeros(n)
    for i in range(net.n_bus):
        if th[i] >= 0: g[th[i]] = gva[0, i]
        if vmx[i] >= 0: g[vmx[i]] = gvm[0, i]
    lam = np.linalg.solve(J.T, g)
    lp, lq, _ = oracle.adjoint_batch(Y, net.bus_type, vm[None], va[None], gva, gvm, method=1)
    for i in range(net.n_bus):
        if th[i] >= 0: assert abs(lp[0, i] - lam[th[i]]) < 1e-11
        if vmx[i] >= 0: assert abs(lq[0, i] - lam[vmx[i]]) < 1e-11


def test_mixed_precision_reference_mode():
    """FP32 linear solves with FP64 residual reach the same tolerance with the same
    or at most one additional iteration."""
    for cfg in (1, 2):
        net = S.make_network(cfg)
        Y = net_Y(net)
        ps, qs, vs = S.make_scenarios(net, batch=8)
        dp = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=1)
        for method in (0, 1):
            mp = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=method, mixed=True)
            assert mp["converged"].all() and np.all(mp["final_norm"] <= 1e-8)
            d = mp["iterations"] - dp["iterations"]
            assert d.min() >= 0 and d.max() <= 1
            np.testing.assert_allclose(mp["vm"], dp["vm"], atol=1e-8)


def test_mixed_precision_inner_refinement():
    """oracle.nr_mixed_ir (SURVEY.md section 8(c) reading 15) pinned to things other than itself: with 0 sweeps it is the C
    oracle's mixed mode (same FP32-rounded solves, so the same iterates); with enough sweeps every linear solve reaches
    FP64 accuracy, so its norm history is that of the FP64 Newton loop (which contains no FP32 arithmetic at all) -- a wrong
    sign, a dropped term or a transposed index in the residual r = -F1 - J1 dz makes the refined step worse than the FP32
    one and fails this; one sweep must already shrink the distance to the FP64 history by orders of magnitude."""
    for cfg in (1, 2):
        net = S.make_network(cfg)
        Y = net_Y(net)
        ps, qs, vs = S.make_scenarios(net, batch=3)
        dp = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=1, want_hist=True)
        mp = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, method=1, mixed=True, want_hist=True)
        for b in range(3):
            r0 = oracle.nr_mixed_ir(Y, net.bus_type, ps[b], qs[b], vs[b], ir_sweeps=0)
            assert r0["iterations"] == mp["iterations"][b] and r0["converged"] == mp["converged"][b]
            np.testing.assert_allclose(r0["vm"], mp["vm"][b], rtol=0, atol=1e-14)
            np.testing.assert_allclose(r0["va"], mp["va"][b], rtol=0, atol=1e-14)
            r3 = oracle.nr_mixed_ir(Y, net.bus_type, ps[b], qs[b], vs[b], ir_sweeps=3)
            k = dp["iterations"][b]
            assert r3["converged"] == 1 and r3["iterations"] == k
            h64, h3, h0 = dp["hist"][b][:k + 1], r3["hist"][:k + 1], r0["hist"][:k + 1]
            assert np.all(np.abs(h3 - h64) <= 1e-6 * h64 + 1e-12)
            np.testing.assert_allclose(r3["vm"], dp["vm"][b], rtol=0, atol=1e-12)
            np.testing.assert_allclose(r3["va"], dp["va"][b], rtol=0, atol=1e-12)
            # the unrefined FP32 loop leaves the FP64 history once the norm is small; one sweep brings it back
            r1 = oracle.nr_mixed_ir(Y, net.bus_type, ps[b], qs[b], vs[b], ir_sweeps=1)
            d0 = np.nanmax(np.abs(h0[:min(k, r0["iterations"]) + 1] - h64[:min(k, r0["iterations"]) + 1]))
            d1 = np.nanmax(np.abs(r1["hist"][:k + 1] - h64))
            assert d1 <= 1e-3 * d0 + 1e-12


def test_recorded_configs_are_feasible():
    """sable_synth.CONFIGS carries the (s_net, kappa) accepted by oracle/feasibility_scan.py."""
    for cfg in (1, 2, 3, 4):
        net = S.make_network(cfg)
        assert net.f.shape[0] == net.cfg.n_branch and (net.bus_type == S.PV).sum() == net.cfg.n_pv
        Y = net_Y(net)
        ps, qs, vs = S.make_scenarios(net, batch=8)
        res = oracle.nr_batch(Y, net.bus_type, ps, qs, vs, max_it=net.cfg.max_it, method=1)
        assert res["converged"].all() and res["iterations"].max() <= 7
