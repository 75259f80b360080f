"""GPU parity at BASELINE.json config 5's two large sizes, 512x512x160 and 512x512x256, element by element against the
oracle at the per-kernel bar |a - b| <= 1e-4 + 1e-5 |b| (north_star).

At these sizes the kernels run shapes no smaller test reaches: four x-blocks per row in the force kernels, 4 x 64
smoother tiles with the even z split crossing many columns, nx / 4 > 64 in the pyramid kernels' grids.  Inputs are
phantoms.sweep_inputs (config 5's recipe).  One oracle call costs 1-20 s of one host core here, so
every case computes its reference, compares on the device and drops it; the file costs about a minute.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

ATOL, RTOL = 1e-4, 1e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


@pytest.fixture(scope="module")
def B(torch_cuda):
    from paper_0909_0928_b200 import build
    build.build()
    from paper_0909_0928_b200 import binding
    binding.lib()
    return binding


def _inputs(dims, seed):
    from paper_0909_0928_b200 import phantoms
    return phantoms.sweep_inputs(dims, seed)


@pytest.fixture(scope="module")
def case160():
    return _inputs((512, 512, 160), 502)


def dev(torch, a):
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def assert_close_dev(torch, gpu, ref_np, what, atol=ATOL):
    """gpu: device tensor; ref_np: the oracle's array.  Compared on the device, every element."""
    ref = dev(torch, ref_np)
    assert gpu.shape == ref.shape, what
    viol = (gpu.double() - ref.double()).abs() - (atol + RTOL * ref.double().abs())
    worst = float(viol.max())
    assert bool(torch.isfinite(gpu).all()), what
    assert worst <= 0, f"{what}: max violation {worst:.3e} at flat index {int(viol.argmax())}"


@pytest.mark.parametrize("variant", [0, 2, 5])
def test_warp_force_512x512x160(torch_cuda, B, oracle, case160, variant):
    torch = torch_cuda
    S, M, u = case160
    dims = (S.shape[2], S.shape[1], S.shape[0])
    ic = variant == 5
    ub = np.ascontiguousarray(-0.5 * u[::-1]) if ic else None        # a backward field that is not -u
    ref_u, ref_ub, ref_m = oracle.warp_force(variant, 1.0, S, M, u, ub)
    eng = B.Demons(dims, variant=variant)
    dS, dM, du = dev(torch, S), dev(torch, M), dev(torch, u)
    dub = dev(torch, ub) if ic else None
    out = torch.full_like(du, float("nan"))
    outb = torch.full_like(du, float("nan")) if ic else None
    met = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    B.demons_warp_force(eng.ctx, dims, dS, dM, du, out, dub, outb, met)
    torch.cuda.synchronize()
    assert_close_dev(torch, out, ref_u, f"warp_force variant {variant} u_out")
    if ic:
        assert_close_dev(torch, outb, ref_ub, "warp_force variant 5 ub_out")
    np.testing.assert_allclose(met.cpu().numpy(), np.asarray(ref_m, dtype=np.float64), rtol=1e-5)
    eng.close()


@pytest.mark.parametrize("sigma", [1.0, 2.0])
def test_smooth_512x512x160(torch_cuda, B, oracle, case160, sigma):
    torch = torch_cuda
    _, _, u = case160
    dims = (u.shape[3], u.shape[2], u.shape[1])
    ref = oracle.smooth(u, sigma)
    eng = B.Demons(dims, variant=0, sigma=sigma)
    du = dev(torch, u)
    out = torch.full_like(du, float("nan"))
    B.demons_smooth(eng.ctx, dims, du, out, 3, sigma)
    torch.cuda.synchronize()
    assert_close_dev(torch, out, ref, f"smooth sigma {sigma}")
    eng.close()


def test_restrict_prolong_512x512x160(torch_cuda, B, oracle, case160):
    torch = torch_cuda
    S, _, u = case160
    dims = (S.shape[2], S.shape[1], S.shape[0])
    eng = B.Demons(dims, variant=0)
    cdims = B.demons_level_dims(eng.ctx, 1)
    ref_c = oracle.restrict(S)
    out_c = torch.full((cdims[2], cdims[1], cdims[0]), float("nan"), dtype=torch.float32, device="cuda:0")
    B.demons_restrict(eng.ctx, dims, dev(torch, S), out_c)
    torch.cuda.synchronize()
    assert_close_dev(torch, out_c, ref_c, "restrict")
    uc = np.stack([oracle.restrict(u[c]) for c in range(3)])           # a coarse field with the fine one's structure
    ref_f = oracle.prolong(uc, S.shape)
    out_f = torch.full((3,) + S.shape, float("nan"), dtype=torch.float32, device="cuda:0")
    B.demons_prolong(eng.ctx, cdims, dev(torch, uc), dims, out_f)
    torch.cuda.synchronize()
    assert_close_dev(torch, out_f, ref_f, "prolong")
    eng.close()


def test_warp_force_and_smooth_512x512x256(torch_cuda, B, oracle):
    """The largest size config 5 names: the passive force pass and the sigma = 1 smoother."""
    torch = torch_cuda
    S, M, u = _inputs((512, 512, 256), 503)
    dims = (512, 512, 256)
    eng = B.Demons(dims, variant=0)
    dS, dM, du = dev(torch, S), dev(torch, M), dev(torch, u)
    out = torch.full_like(du, float("nan"))
    met = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    B.demons_warp_force(eng.ctx, dims, dS, dM, du, out, None, None, met)
    torch.cuda.synchronize()
    ref_u, _, ref_m = oracle.warp_force(0, 1.0, S, M, u, None)
    assert_close_dev(torch, out, ref_u, "warp_force 512x512x256")
    np.testing.assert_allclose(met.cpu().numpy(), np.asarray(ref_m, dtype=np.float64), rtol=1e-5)
    del ref_u
    B.demons_smooth(eng.ctx, dims, du, out, 3, 1.0)
    torch.cuda.synchronize()
    assert_close_dev(torch, out, oracle.smooth(u, 1.0), "smooth 512x512x256 sigma 1")
    eng.close()
