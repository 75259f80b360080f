"""demons_ssd_static: the SSD for callers who may not allocate device memory.

Who needs it: code that is handed device pointers by somebody else and must leave device memory as it found it -- a
checking hook inside a planning system, a plug-in whose host application owns the memory budget and forbids cudaMalloc,
a loop that cannot afford the device-wide stall of an allocator call.  Those callers cannot build the workspace that
demons_ssd wants, so this entry point keeps its scratch (block partials + a counter) in a fixed array inside
libdemons.so and refuses volumes that array cannot serve (more than 2^26 voxels).

What is checked here: the result equals demons_ssd's (the existing, workspace-based path, itself checked against the
oracle in test_gpu_parity.py) at the 1e-5 relative tolerance this suite uses for reductions, on calls made back to back
on one stream with no synchronisation between them -- a large volume first, a smaller one second, so that partial sums
left in the shared array by the first call would show up in the second -- and that the first call repeated gives the
same bits.  This file sorts last on purpose: `pytest -x` stops at the first failure, and nothing should hide behind a
failure here.  It uses no state of the other test files, so it passes alone in a fresh process as well.
"""

import numpy as np
import pytest


@pytest.fixture(scope="module")
def B():
    from paper_0909_0928_b200 import build
    build.build()
    from paper_0909_0928_b200 import binding
    binding.lib()
    return binding


def test_static_ssd_refuses_what_its_scratch_cannot_serve(B):
    """Host-side checks come before any CUDA call, so they run without a GPU: a volume beyond the limit is refused with
    a message that names the limit, and so are NULL pointers and bad dims.  The pointers are never dereferenced."""
    fake = 4096
    with pytest.raises(B.DemonsError) as e:
        B.demons_ssd_static((512, 512, 257), fake, fake, fake, None, fake)
    assert e.value.code == B.E_UNSUPPORTED
    assert str(B.SSD_STATIC_MAX_VOXELS) in str(e.value) and "demons_ssd" in str(e.value)
    assert B.SSD_STATIC_MAX_VOXELS == 512 * 512 * 256
    for dims, args in [((0, 4, 4), (fake, fake, fake, None, fake)), ((4, 4, 4), (None, fake, fake, None, fake)),
                       ((4, 4, 4), (fake, fake, None, None, fake)), ((4, 4, 4), (fake, fake, fake, None, None))]:
        with pytest.raises(B.DemonsError) as e:
            B.demons_ssd_static(dims, *args)
        assert e.value.code == B.E_ARG
    assert B.lib().demons_ssd_static(None, fake, fake, fake, None, fake, None) == B.E_ARG


def _case(P, dims, seed):
    rng = np.random.default_rng(seed)
    S = P.blob_volume(dims, rng, 20, 10.0)
    M = P.resample(S, P.bump_field(dims, rng, 4, (4.0, 10.0), 3.0))
    u = P.bump_field(dims, rng, 6, (3.0, 9.0), 3.0, centre_frac=1.0)
    ub = P.bump_field(dims, rng, 6, (3.0, 9.0), 3.0, centre_frac=1.0)
    return S, M, u, ub


@pytest.mark.gpu
@pytest.mark.parametrize("two_field", [False, True])
def test_static_ssd_equals_workspace_ssd_on_calls_in_a_row(B, two_field):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_0909_0928_b200 import phantoms as P

    def dev(a):
        return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")

    # 31 blocks of 4096 voxels with a ragged last one, then 9 blocks: the second call reuses the array the first filled
    cases = [((136, 44, 21), 71), ((44, 36, 22), 72)]
    variant = B.INVERSE_CONSISTENT if two_field else B.PASSIVE
    bufs, want = [], []
    for dims, seed in cases:
        S, M, u, ub = (dev(a) for a in _case(P, dims, seed))
        bufs.append((dims, S, M, u, ub if two_field else None))
        eng = B.Demons(dims, variant=variant)  # the existing path: context + torch-allocated workspace
        ref = torch.zeros(1, dtype=torch.float64, device="cuda:0")
        B.demons_ssd(eng.ctx, dims, S, M, u, ub if two_field else None, ref)
        torch.cuda.synchronize()
        want.append(float(ref[0]))
        eng.close()
    assert all(w > 0 for w in want)

    got = torch.full((3,), -1.0, dtype=torch.float64, device="cuda:0")
    stream = torch.cuda.current_stream()
    order = [0, 1, 0]
    free_after_first = None
    for slot, k in enumerate(order):  # back to back on one stream, nothing in between
        dims, S, M, u, ub = bufs[k]
        B.demons_ssd_static(dims, S, M, u, ub, got[slot:], stream)
        if free_after_first is None:  # the first call may load the kernel's module; later calls must cost no memory
            free_after_first = torch.cuda.mem_get_info()[0]
    assert torch.cuda.mem_get_info()[0] == free_after_first
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    for slot, k in enumerate(order):
        assert abs(got[slot] - want[k]) <= 1e-5 * want[k], (slot, got[slot], want[k])
    assert got[0] == got[2]  # same inputs, same bits: the shared array carries nothing from call to call
