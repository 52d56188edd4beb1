"""GPU parity of the shared-memory-window stencil kernel (csrc/dslash_win.cu) against the fp64 oracle.

The window kernel only runs on lattices whose (z, t) strips are whole 64-site tiles (X/2 * Y % 64 == 0), which
none of the small lattices of test_gpu_parity.py are; here it is forced (bkr_set_dslash_variant) on lattices that span
one, two, three and eight tiles per strip, window reaches of 1, 2 and 3 chunks, cluster sizes 1-4 (fp64: 8 rhs per
CTA, fp32: 16) and ragged N.  Every case checks bkr_dslash_variant() so that a silent fall-back to the plain kernel
cannot pass for the window kernel.  Definition: PAPER.md:95-101 (eq. 2), U1; tolerance DESIGN.md U17.
"""
import numpy as np
import pytest
import torch

from tests import helpers as H

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-13, 1e-5

LATTICES = {
    "16x8x4x4": (16, 8, 4, 4),      # one tile per strip, every y-neighbour wraps inside the window
    "16x16x4x6": (16, 16, 4, 6),    # two tiles per strip, reach 1 chunk
    "8x16x6x4": (8, 16, 6, 4),      # X/2 = 4: four rows per chunk
    "32x8x4x4": (32, 8, 4, 4),      # reach 2 chunks, strip shorter than the window
    "32x32x4x8": (32, 32, 4, 8),    # 8 tiles per strip, the shape of configs 3 and 5
    "48x16x4x4": (48, 16, 4, 4),    # X/2 = 24: tiles start mid-row (x hops reach below the tile), reach 3 chunks: config 4
}


def _round32(a):
    return a.astype(np.complex64).astype(np.complex128)


@pytest.fixture(scope="module", params=sorted(LATTICES))
def lat(request):
    from paper_1710_09745_b200 import binding
    dims = LATTICES[request.param]
    fat, lng = H.np_links(dims, "random", seed=41)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda(), also_f32=True)
    ctx.set_dslash_variant(1)
    return dims, fat, lng, ctx


@pytest.mark.parametrize("N", [7, 8, 11, 16, 24, 32])
def test_window_dslash_fp64(lat, N):
    import oracle
    dims, fat, lng, ctx = lat
    for parity in (0, 1):
        v = H.np_sources(dims, N, 900 + N + parity)
        got = ctx.dslash_canonical(parity, torch.from_numpy(v).cuda()).cpu().numpy()
        assert ctx.dslash_variant() == 1
        assert H.relerr_inf(got, oracle.dslash(dims, fat, lng, parity, v)) <= TOL64


@pytest.mark.parametrize("N", [13, 16, 32])
def test_window_dslash_fp32(lat, N):
    import oracle
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat
    v = _round32(H.np_sources(dims, N, 950 + N))
    got = ctx.dslash_canonical(1, torch.from_numpy(v).cuda(), binding.F32).cpu().numpy()
    assert ctx.dslash_variant() == 1
    assert H.relerr_inf(got, oracle.dslash(dims, _round32(fat), _round32(lng), 1, v)) <= TOL32


@pytest.mark.parametrize("N", [8, 16])
def test_window_apply_M_xpay_epilogue(lat, N):
    """second half of M = 4 m^2 - D_eo D_oe runs the a * xp - D epilogue of the window kernel"""
    import oracle
    dims, fat, lng, ctx = lat
    v = H.np_sources(dims, N, 980 + N)
    got = ctx.apply_M_canonical(0.05, torch.from_numpy(v).cuda()).cpu().numpy()
    assert ctx.dslash_variant() == 1
    assert H.relerr_inf(got, oracle.apply_M(dims, fat, lng, 0.05, v)) <= TOL64


def test_window_matches_plain_kernel_bitwise_inputs(lat):
    """the two kernels sum the 16 hops in different orders: they agree to rounding, not bit for bit, and the
    automatic choice must give one of the two"""
    dims, fat, lng, ctx = lat
    v = torch.from_numpy(H.np_sources(dims, 16, 77)).cuda()
    try:
        ctx.set_dslash_variant(0)
        plain = ctx.dslash_canonical(0, v)
        assert ctx.dslash_variant() == 0
        ctx.set_dslash_variant(1)
        win = ctx.dslash_canonical(0, v)
        assert ctx.dslash_variant() == 1
        assert float((plain - win).abs().max() / plain.abs().max()) <= 1e-14
        ctx.set_dslash_variant(-1)
        auto = ctx.dslash_canonical(0, v)
        assert torch.equal(auto, win) or torch.equal(auto, plain)
    finally:
        ctx.set_dslash_variant(1)


def test_window_falls_back_when_strip_is_not_whole_tiles():
    from paper_1710_09745_b200 import binding
    import oracle
    dims = (4, 6, 8, 10)
    fat, lng = H.np_links(dims, "random", seed=43)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda())
    ctx.set_dslash_variant(1)
    v = H.np_sources(dims, 8, 5)
    got = ctx.dslash_canonical(0, torch.from_numpy(v).cuda()).cpu().numpy()
    assert ctx.dslash_variant() == 0
    assert H.relerr_inf(got, oracle.dslash(dims, fat, lng, 0, v)) <= TOL64
