"""Cases for compute-sanitizer (memcheck / racecheck / synccheck); not collected by pytest.

  compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
  compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
  compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Configs 1-3 in every placement / slot-group layout of the NR kernel (on chip with and without the level-blob ring, HBM
workspace with and without the dense top front, group sizes 1 / 4 / 8, a team of two CTAs per group), fused and staged
mode, keep_factors on and off, FP64 and mixed, with a ragged last group and one scenario that does not converge (so the
spare workspace group that absorbs the stores of finished slots is live), followed by the adjoint, the recovery and the
layer backward on the kept factors.  Results are checked for convergence only (parity is tests/test_gpu_parity.py).
"""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2606_07099_b200 as sb  # noqa: E402
import sable_synth as S  # noqa: E402


def run(cfg, batch, mode=sb.FUSED, precision=sb.FP64, keep=True, **tune):
    net = S.make_network(cfg)
    c = net.cfg
    Y = S.ybus_triplets(net.n_bus, net.f, net.t, net.r, net.x, net.b)
    ps, qs, vs = S.make_scenarios(net, batch=batch)
    ps[min(7, batch - 1)] *= 30.0                    # one scenario that does not converge
    gva, gvm = S.make_adjoint_rhs(net, batch=batch)
    d = lambda a: torch.from_numpy(a).cuda()
    ctx = sb.Context(net.n_bus, *Y, net.bus_type, net.slack, max_batch=batch + 5, mode=mode, precision=precision,
                     keep_factors=keep, **tune)
    out = ctx.solve(d(ps), d(qs), d(vs), tol=c.tol, max_it=12)
    if keep:
        ctx.adjoint(d(gva), d(gvm))
        ctx.layer_backward(out["vm"], out["va"], d(gva), d(gvm), d(gvm), d(gva))
        ctx.adjoint_refined(out["vm"], out["va"], d(gva), d(gvm), sweeps=1)
    ctx.recover(out["vm"], out["va"])
    ctx.pivot_flags(batch)
    torch.cuda.synchronize()
    conv = int(out["converged"].sum().item())
    info = ctx.info
    print(f"cfg {cfg} batch {batch} mode {mode} precision {precision} keep {keep} {tune}: placement {info['placement']} G {info['slots_per_cta']} "
          f"threads {info['threads']} cluster {info['cluster']} front {info['front_k']}: converged {conv}/{batch}", flush=True)
    assert conv >= batch - 1
    ctx.close()


def main():
    run(1, 21)
    run(1, 21, mode=sb.STAGED)
    run(2, 43, group=4, on_chip=1)
    run(2, 43, group=2, on_chip=1, ring_slots=2, ring_slot_bytes=4096)
    run(2, 43, group=8, on_chip=1, keep=False)
    run(2, 43, group=1, on_chip=0, front_nodes=0)
    run(2, 43, group=4, on_chip=0, front_nodes=13, front_kb=64)
    run(2, 43, group=4, on_chip=0, front_nodes=13, front_kb=64, precision=sb.MIXED)
    run(2, 43, group=2, on_chip=0, cluster=2)
    run(2, 43, group=4, on_chip=0, mode=sb.STAGED)
    run(3, 37, group=4, on_chip=0)
    run(3, 37, group=1, on_chip=0, threads=256, front_nodes=9, front_kb=64, keep=False)
    run(3, 19, group=8, on_chip=0, threads=256, precision=sb.MIXED)
    run(3, 19, group=4, on_chip=0, cluster=2, threads=256)
    # merged single-wave layouts: 4 / 16 scenarios per CTA of 768 / 1 024 threads, FP64 and FP32 pair records
    run(2, 43, group=4, on_chip=0, threads=768)
    run(3, 37, group=16, on_chip=0, threads=1024, precision=sb.MIXED)
    run(3, 37, group=16, on_chip=0, threads=1024, keep=False)
    print("sanitizer cases done")


if __name__ == "__main__":
    main()
