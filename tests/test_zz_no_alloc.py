"""wz_apply_MdagM_noalloc (include/wz.h): the matvec without a plan and without device allocation, its scratch in a
static device array inside libwz.so.  Checked against the existing path (a plan's wz_apply_MdagM) on two calls in a
row, within the tolerances of tests/test_gpu_parity.py.  This file sorts last on purpose (the suite runs with
pytest -x); it must pass alone in a fresh process and after the other tests."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

TOL = {"c128": 1e-12, "c64": 2e-5}
NPDT = {"c128": np.complex128, "c64": np.complex64}


def rel(a, ref):
    return float(np.linalg.norm((a - ref).ravel()) / np.linalg.norm(ref.ravel()))


@pytest.fixture(scope="module")
def wz():
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device")
    from paper_1005_3276_b200 import wz as _wz

    _wz.lib()
    return _wz


@pytest.mark.parametrize("dims,dtype,nsrc", [((8, 8, 8, 8), "c128", 2), ((16, 16, 16, 16), "c64", 1),
                                             ((8, 4, 16, 8), "c64", 3)])
def test_noalloc_matvec_equals_plan_matvec_twice_in_a_row(wz, dims, dtype, nsrc):
    from paper_1005_3276_b200 import inputs

    m, g, rho = 0.05 + 0.02j, 1.0 - 0.3j, 1.0
    phi = torch.from_numpy(inputs.make_phi(21, dims, 0.4, NPDT[dtype])).cuda()
    b1 = torch.from_numpy(inputs.make_sources(21, nsrc, dims, NPDT[dtype])).cuda()
    b2 = torch.from_numpy(inputs.make_sources(22, nsrc, dims, NPDT[dtype])).cuda()
    plan = wz.Plan(dims, dtype, nsrc)
    ref1 = plan.apply_MdagM(phi, b1, m, g, rho).cpu().numpy()
    ref2 = plan.apply_MdagM(phi, b2, m, g, rho).cpu().numpy()
    out1, out2 = torch.empty_like(b1), torch.empty_like(b2)
    # two calls in a row on one stream, no synchronisation in between: the second reuses the static scratch the
    # first left behind
    wz.apply_MdagM_noalloc(phi, b1, m, g, rho, out=out1)
    wz.apply_MdagM_noalloc(phi, b2, m, g, rho, out=out2)
    torch.cuda.synchronize()
    assert rel(out1.cpu().numpy(), ref1) <= TOL[dtype]
    assert rel(out2.cpu().numpy(), ref2) <= TOL[dtype]
    # a third call on the first input reproduces the first, and the driver's free memory does not move across it
    out3 = torch.empty_like(b1)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    wz.apply_MdagM_noalloc(phi, b1, m, g, rho, out=out3)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info()[0]
    assert torch.equal(out3, out1)
    assert free_after >= free_before, (free_before, free_after)


def test_noalloc_rejects_what_does_not_fit(wz):
    from paper_1005_3276_b200 import inputs

    dims = (16, 16, 16, 16)  # one complex128 source needs 2 x 4 MiB = the whole array: fits; two do not
    phi = torch.from_numpy(inputs.make_phi(21, dims, 0.4)).cuda()
    b = torch.from_numpy(inputs.make_sources(21, 2, dims)).cuda()
    out = torch.empty_like(b)
    with pytest.raises(wz.WZError) as e:
        wz.apply_MdagM_noalloc(phi, b, 0.05, 1.0, 1.0, out=out)
    assert e.value.status == wz.WZ_EINVAL and "WZ_NOALLOC_MAX_BYTES" in str(e.value)
    one = wz.apply_MdagM_noalloc(phi, b[:1].contiguous(), 0.05, 1.0, 1.0)
    ref = wz.Plan(dims, "c128", 1).apply_MdagM(phi, b[:1].contiguous(), 0.05, 1.0, 1.0)
    assert rel(one.cpu().numpy(), ref.cpu().numpy()) <= TOL["c128"]
    with pytest.raises(wz.WZError) as e:  # T odd
        wz.apply_MdagM_noalloc(torch.zeros((5, 4, 4, 4), dtype=torch.complex128, device="cuda"),
                               torch.zeros((4, 5, 4, 4, 4), dtype=torch.complex128, device="cuda"), 0.05, 1.0)
    assert e.value.status == wz.WZ_EINVAL
