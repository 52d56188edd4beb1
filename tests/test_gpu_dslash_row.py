"""GPU parity of the row-window stencil kernel (csrc/dslash_row.cu) against the fp64 oracle.

The kernel holds up to 16 rhs per CTA (17-32: a cluster of two CTAs with multicast links), takes its x/y neighbours
from a shared-memory window of whole x-rows and its z/t neighbours by register loads two hops ahead.  It is not in the
automatic choice, so every case forces it with bkr_set_dslash_variant(2) and checks
bkr_dslash_variant() afterwards: a silent fall-back cannot pass.  Lattices: X = 32 (the only row length it is built
for) with 2, 1 and 8 tiles per strip, strips shorter than the window (Y = 4, 8: every y hop wraps inside it), work
units of 1, 2 and all tiles of a strip, ragged N on both sides of the cluster boundary.
Definition: PAPER.md:95-101 (eq. 2), U1; tolerance DESIGN.md U17.
"""
import pytest
import torch

from tests import helpers as H

pytestmark = pytest.mark.gpu

TOL64 = 1e-13
LATTICES = {"32x8x4x4": (32, 8, 4, 4), "32x4x4x6": (32, 4, 4, 6), "32x32x4x8": (32, 32, 4, 8)}


@pytest.fixture(scope="module", params=sorted(LATTICES))
def lat(request):
    from paper_1710_09745_b200 import binding
    dims = LATTICES[request.param]
    fat, lng = H.np_links(dims, "random", seed=47)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda())
    ctx.set_dslash_variant(2)
    return dims, fat, lng, ctx


@pytest.mark.parametrize("N", [5, 9, 12, 13, 16, 17, 24, 29, 32])
def test_row_dslash_fp64(lat, N):
    import oracle
    dims, fat, lng, ctx = lat
    for parity in (0, 1):
        v = H.np_sources(dims, N, 700 + N + parity)
        got = ctx.dslash_canonical(parity, torch.from_numpy(v).cuda()).cpu().numpy()
        assert ctx.dslash_variant() == 2
        assert H.relerr_inf(got, oracle.dslash(dims, fat, lng, parity, v)) <= TOL64


@pytest.mark.parametrize("N", [11, 16, 32])
@pytest.mark.parametrize("unit_tiles", [1, 2, 8])
def test_row_apply_M_xpay_epilogue_and_units(lat, N, unit_tiles):
    """second half of M = 4 m^2 - D_eo D_oe runs the a * xp - D epilogue; work units of 1, 2 and all tiles
    of a strip change the window prologue and the cross-tile prefetch of the z/t neighbours"""
    import oracle
    from paper_1710_09745_b200 import binding
    dims, fat, lng, ctx = lat
    ctx.set_option(binding.OPT_ROW_UNIT_TILES, unit_tiles)
    try:
        v = H.np_sources(dims, N, 780 + N)
        got = ctx.apply_M_canonical(0.05, torch.from_numpy(v).cuda()).cpu().numpy()
        assert ctx.dslash_variant() == 2
        assert H.relerr_inf(got, oracle.apply_M(dims, fat, lng, 0.05, v)) <= TOL64
    finally:
        ctx.set_option(binding.OPT_ROW_UNIT_TILES, 0)


def test_row_falls_back_when_x_is_not_32():
    import oracle
    from paper_1710_09745_b200 import binding
    dims = (16, 16, 4, 6)
    fat, lng = H.np_links(dims, "random", seed=49)
    ctx = binding.Context(dims)
    ctx.load_links(torch.from_numpy(fat).cuda(), torch.from_numpy(lng).cuda())
    ctx.set_dslash_variant(2)
    v = H.np_sources(dims, 16, 6)
    got = ctx.dslash_canonical(0, torch.from_numpy(v).cuda()).cpu().numpy()
    assert ctx.dslash_variant() == 0
    assert H.relerr_inf(got, oracle.dslash(dims, fat, lng, 0, v)) <= TOL64
