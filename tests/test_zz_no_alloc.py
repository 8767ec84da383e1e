"""The allocation-free entry point sable_injections_static (include/sable.h, csrc/sable_static.cu): its scratch is a static
device array shared by every call, so the checks run two calls in a row -- the second on a different, smaller batch whose
slices overlap what the first call left in the array -- and compare each with the existing path (sable_recover on a
context) within the tolerance the recovery tests use (1e-13 of the row scale).  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

import sable_synth as S
from util import dev, make_ctx, random_state

pytestmark = pytest.mark.gpu


def _row_scale(Yt, vm):
    """sum_k |Y_ik| |V_k| |V_i| per bus from the harness-side triplets: the magnitude the rounding error scales with."""
    row_ptr, col, g, b = Yt
    rows = np.repeat(np.arange(len(row_ptr) - 1), np.diff(row_ptr))
    sc = np.zeros_like(vm)
    for bb in range(vm.shape[0]):
        np.add.at(sc[bb], rows, np.hypot(g, b) * vm[bb, col])
    return np.maximum(sc * vm, 1.0)


def _device_csr(Yt):
    row_ptr, col, g, b = Yt
    return dev(row_ptr.astype(np.int32)), dev(col.astype(np.int32)), dev(g), dev(b)


@pytest.mark.parametrize("cfg,batch", [(3, 64), (5, 6)])
def test_injections_static_matches_recover_twice(cfg, batch):
    import torch
    import paper_2606_07099_b200 as sb
    net = S.make_network(cfg)
    Yt = S.ybus_triplets(net.n_bus, net.f, net.t, net.r, net.x, net.b)
    csr = _device_csr(Yt)
    ctx = make_ctx(net, max_batch=batch, keep_factors=False)
    # set-up call (batch 0): looks up the array's address for this device, launches nothing
    empty = torch.empty((0, net.n_bus), dtype=torch.float64, device="cuda")
    sb.injections_static(*csr, empty, empty, out=(empty, empty))
    for call, (nb, seed) in enumerate([(batch, 11), (max(1, batch // 3), 12)]):
        vm, va = random_state(net, nb, seed)
        d_vm, d_va = dev(vm), dev(va)
        out = (torch.full_like(d_vm, float("nan")), torch.full_like(d_vm, float("nan")))
        p_new, q_new = sb.injections_static(*csr, d_vm, d_va, out=out)
        p_old, q_old = ctx.recover(d_vm, d_va)
        torch.cuda.synchronize()
        sc = _row_scale(Yt, vm)
        dp = np.abs(p_new.cpu().numpy() - p_old.cpu().numpy())
        dq = np.abs(q_new.cpu().numpy() - q_old.cpu().numpy())
        assert np.isfinite(p_new.cpu().numpy()).all() and np.isfinite(q_new.cpu().numpy()).all()
        assert (dp <= 1e-13 * sc).all(), f"call {call}: max P difference {dp.max()}"
        assert (dq <= 1e-13 * sc).all(), f"call {call}: max Q difference {dq.max()}"
    ctx.close()


def test_injections_static_rejects_oversize():
    import torch
    import paper_2606_07099_b200 as sb
    net = S.make_network(3)
    Yt = S.ybus_triplets(net.n_bus, net.f, net.t, net.r, net.x, net.b)
    csr = _device_csr(Yt)
    batch = sb.STATIC_SCRATCH_BYTES // (16 * net.n_bus) + 1          # one scenario beyond the array
    vm = torch.ones((batch, net.n_bus), dtype=torch.float64, device="cuda")
    va = torch.zeros_like(vm)
    with pytest.raises(sb.SableError) as ei:
        sb.injections_static(*csr, vm, va)
    assert ei.value.status == 1 and "static scratch" in str(ei.value)
    # the largest batch that fits still runs
    p, q = sb.injections_static(*csr, vm[:batch - 1], va[:batch - 1])
    torch.cuda.synchronize()
    assert torch.isfinite(p).all() and torch.isfinite(q).all()
