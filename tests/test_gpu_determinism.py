"""Bit-exact rerun test of the window stencil (round 2): a launch that reads a ring slot after its refill has landed gives a
result that differs from run to run.  The round-2 kernel first released a slot right after issuing its last loads; with the
xpay loads congesting the load queue, 2e-4 of the launches on this lattice (16^4, where a refill is ~700 cycles away) read one
32-byte sector of hop 8's operands from hop 11's chunk -- invisible to any single parity comparison.  20 000 launches would have
shown ~4 mismatches; the fix (a CTA-scope fence in front of every slot release) shows none in 2 x 10^6."""
import pytest
import torch

import oracle
from tests import helpers as H

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,N,prec,launches", [((16, 16, 16, 16), 8, "f64", 20000), ((16, 16, 16, 16), 16, "f64", 6000),
                                                 ((16, 16, 16, 16), 16, "f32", 10000), ((16, 8, 4, 4), 8, "f64", 20000)])
def test_window_stencil_reruns_are_bit_identical(dims, N, prec, launches):
    from paper_1710_09745_b200 import binding
    pr = binding.F64 if prec == "f64" else binding.F32
    fat, lng = H.np_links(dims, "perturbed", seed=77)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    ctx.set_dslash_variant(1)
    a, xp = ctx.empty_native(N, pr).normal_(), ctx.empty_native(N, pr).normal_()
    ref, refx, out = ctx.empty_native(N, pr), ctx.empty_native(N, pr), ctx.empty_native(N, pr)
    ctx.dslash(1, N, a, ref, pr)
    assert ctx.dslash_variant() == 1
    ctx.dslash_xpay(0, N, 0.37, xp, a, refx, pr)
    # the reference launches themselves against the oracle (the rest only has to repeat them bit for bit)
    an = ctx.unpack(a, N, pr).cpu().numpy()
    want = oracle.dslash(dims, fat, lng, 1, an)
    got = ctx.unpack(ref, N, pr).cpu().numpy()
    assert abs(got - want).max() <= (1e-13 if prec == "f64" else 1e-5) * abs(want).max()
    ity = torch.int64 if prec == "f64" else torch.int32
    bad = torch.zeros(2, dtype=torch.int64, device="cuda")
    for _ in range(launches):
        ctx.dslash_xpay(0, N, 0.37, xp, a, out, pr)
        bad[0] += (out.view(ity) != refx.view(ity)).any()
    for _ in range(launches // 4):
        ctx.dslash(1, N, a, out, pr)
        bad[1] += (out.view(ity) != ref.view(ity)).any()
    assert bad.tolist() == [0, 0]
