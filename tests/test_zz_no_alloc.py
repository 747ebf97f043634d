"""srp_forces_noalloc (include/srp.h): the forces call that allocates nothing -- its scratch is a static device array
of the library -- against srp_forces on the same designs, directions and seed.  Collected last (file name), so that
with `pytest -x` a failure here hides no other test; passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

from paper_2602_10712_b200 import workloads as W

pytestmark = pytest.mark.gpu

NOALLOC_MAX_PAIRS = 65536


@pytest.fixture()
def ctx():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2602_10712_b200.binding import Context
    c = Context(0)
    yield c
    c.close()


def cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a, np.float32)).cuda()


def test_noalloc_forces_equal_srp_forces_twice_in_a_row(ctx):
    """Two calls in a row on different inputs (the second finds the first one's sums in the shared array) and a third
    on a design with a BVH traced ray by ray; each against srp_forces.  The sums are order-independent int64 fixed
    point, so the two paths agree to the bit; the bound written here is the 1e-6 relative L2 of the reproducibility
    tests."""
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 24))
    sun_a, sun_b = cuda(W.fibonacci_sphere(16)), cuda(W.fibonacci_sphere(7)[::-1].copy())
    ref_a = ctx.srp_forces(dz, sun_a, 1 << 14, 4, 3).cpu().numpy()
    ref_b = ctx.srp_forces(dz, sun_b, 1 << 12, 2, 9).cpu().numpy()
    out_a = torch.full((24, 16, 3), float("nan"), dtype=torch.float32, device="cuda")
    out_b = torch.full((24, 7, 3), float("nan"), dtype=torch.float32, device="cuda")
    torch.cuda.synchronize()
    before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    ctx.srp_forces_noalloc(dz, sun_a, 1 << 14, 4, 3, out_a)
    ctx.srp_forces_noalloc(dz, sun_b, 1 << 12, 2, 9, out_b)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before and torch.cuda.mem_get_info()[0] >= free_before   # nothing allocated
    for got, ref in ((out_a.cpu().numpy(), ref_a), (out_b.cpu().numpy(), ref_b)):
        assert np.isfinite(got).all() and np.linalg.norm(ref) > 0
        assert np.linalg.norm(got - ref) <= 1e-6 * np.linalg.norm(ref)
    # the same pair of calls again: nothing of the earlier calls is left in the array
    ctx.srp_forces_noalloc(dz, sun_a, 1 << 14, 4, 3, out_a)
    assert np.array_equal(out_a.cpu().numpy(), ref_a)
    dz.free()

    # a design with a hierarchy, about one ray per triangle or fewer: per-ray traversal, no ray queue
    big = ctx.srp_build_designs(W.FAMILY_DETAILED, W.draw_params(W.FAMILY_DETAILED, 1))
    sun = cuda(W.fibonacci_sphere(3))
    ref = ctx.srp_forces(big, sun, 1 << 14, 3, 1).cpu().numpy()
    out = torch.empty((1, 3, 3), dtype=torch.float32, device="cuda")
    ctx.srp_forces_noalloc(big, sun, 1 << 14, 3, 1, out)
    got = out.cpu().numpy()
    assert np.linalg.norm(got - ref) <= 1e-6 * np.linalg.norm(ref)
    big.free()


def test_noalloc_limits_are_errors(ctx):
    from paper_2602_10712_b200.binding import SrpError
    dz = ctx.srp_build_designs(W.FAMILY_BOXWING, W.draw_params(W.FAMILY_BOXWING, 257))
    sun = cuda(W.fibonacci_sphere(256))                       # 257 x 256 = 65792 pairs > 65536
    out = torch.empty((257, 256, 3), dtype=torch.float32, device="cuda")
    with pytest.raises(SrpError) as e:
        ctx.srp_forces_noalloc(dz, sun, 1 << 10, 2, 0, out)
    assert e.value.status == -1 and "SRP_NOALLOC_MAX_PAIRS" in str(e.value)
    ok = ctx.srp_forces_noalloc(dz, sun[:255], 1 << 10, 2, 0, out[:, :255].contiguous())     # 65535 pairs
    assert torch.isfinite(ok).all()
    dz.free()
    big = ctx.srp_build_designs(W.FAMILY_DETAILED, W.draw_params(W.FAMILY_DETAILED, 1))
    out = torch.empty((1, 2, 3), dtype=torch.float32, device="cuda")
    with pytest.raises(SrpError) as e:                        # 2^20 rays on 49 840 triangles: beams and a ray queue
        ctx.srp_forces_noalloc(big, cuda(W.fibonacci_sphere(2)), 1 << 20, 2, 0, out)
    assert e.value.status == -4
    big.free()
