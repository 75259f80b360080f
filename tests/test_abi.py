"""CPU-side checks of the C-ABI library: it loads, exports every symbol include/demons.h declares,
its host-only entry points work, and its compute entry points fail loudly (no CPU fallback)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_0909_0928_b200 import build
    build.build()
    from paper_0909_0928_b200 import binding
    binding.lib()
    return binding


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "demons.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(demons_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_exported(B):
    names = _declared_functions()
    assert len(names) >= 15
    L = ctypes.CDLL(B.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/demons.h but not exported"
    # and the binding mirrors the header one to one
    assert sorted(B.SIGNATURES) == names
    for n in names:
        assert callable(getattr(B, n))


def test_create_validates_arguments(B):
    ok = B.demons_create((64, 64, 32), (1, 1, 1), B.PASSIVE, 1.0, 1.0)
    B.demons_destroy(ok)
    bad = [
        dict(dims=(0, 64, 32)), dict(dims=(64, 64, 1 << 20)), dict(spacing=(1, 0, 1)), dict(variant=6),
        dict(variant=-1), dict(alpha=0.0), dict(sigma=0.0), dict(sigma=-1.0),
    ]
    for kw in bad:
        args = dict(dims=(64, 64, 32), spacing=(1, 1, 1), variant=0, alpha=1.0, sigma=1.0)
        args.update(kw)
        with pytest.raises(B.DemonsError) as e:
            B.demons_create(**args)
        assert e.value.code == B.E_ARG
    with pytest.raises(B.DemonsError) as e:
        B.demons_create((64, 64, 32), (1, 1, 1), 0, 1.0, 11.0)  # R = 33 > DEMONS_MAX_RADIUS
    assert e.value.code == B.E_UNSUPPORTED


def test_level_dims_and_workspace_size(B):
    ctx = B.demons_create((256, 256, 110), (0.97, 0.97, 2.5), B.INVERSE_CONSISTENT, 1.0, 1.0)
    # ceil rule, reading A12: 110 -> 55 -> 28
    assert B.demons_level_dims(ctx, 0) == (256, 256, 110)
    assert B.demons_level_dims(ctx, 1) == (128, 128, 55)
    assert B.demons_level_dims(ctx, 2) == (64, 64, 28)
    w1, w3 = B.demons_workspace_bytes(ctx, 1), B.demons_workspace_bytes(ctx, 3)
    N = 256 * 256 * 110
    assert w3 > w1 > 17 * N * 4  # 2 warped images, 2 updates, tmp, staging of S, M, u, ub
    assert B.demons_workspace_bytes(ctx, 0) == 0 and B.demons_workspace_bytes(ctx, 9) == 0
    B.demons_destroy(ctx)


def test_no_cpu_fallback(B):
    """Without a CUDA device every compute entry point must fail with DEMONS_E_CUDA / E_WORKSPACE,
    never compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    ctx = B.demons_create((8, 8, 8), (1, 1, 1), 0, 1.0, 1.0)
    with pytest.raises(B.DemonsError) as e:
        B.demons_set_workspace(ctx, 256 * 4096, 1 << 30)
    assert e.value.code == B.E_CUDA
    import numpy as np
    a = np.zeros((3, 8, 8, 8), np.float32)
    b = np.zeros_like(a)
    with pytest.raises(B.DemonsError) as e:
        B.demons_smooth(ctx, (8, 8, 8), a, b, 3, 1.0)
    assert e.value.code == B.E_WORKSPACE  # no workspace could be set, nothing ran
    assert np.all(b == 0)
    B.demons_destroy(ctx)


def test_binding_fails_loudly_without_library(B, tmp_path, monkeypatch):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", str(tmp_path / "missing.so"))
    with pytest.raises(ImportError):
        B.lib()


def test_options_are_host_only_and_validated(B):
    """demons_set_option needs no device: every documented name is accepted, anything else is an error."""
    ctx = B.demons_create((16, 12, 8), (1.0, 1.0, 1.0), B.PASSIVE, 1.0, 1.0)
    try:
        for name in ("graphs", "texture", "generic_smooth", "profile", "l2_persist"):
            B.demons_set_option(ctx, name, 0)
            B.demons_set_option(ctx, name, 1)
        B.demons_set_option(ctx, "texture", 0)
        B.demons_set_option(ctx, "profile", 0)
        with pytest.raises(B.DemonsError):
            B.demons_set_option(ctx, "no_such_option", 1)
    finally:
        B.demons_destroy(ctx)


def test_batch_and_slab_arguments_validated(B):
    """Host-side validation of the batched and the z-slab entry points (no device needed)."""
    import numpy as np
    dims = (16, 12, 10)
    ctx = B.demons_create(dims, (1.0, 1.0, 1.0), B.PASSIVE, 1.0, 1.0)
    try:
        w1, w4 = B.demons_workspace_bytes_batch(ctx, 2, 1), B.demons_workspace_bytes_batch(ctx, 2, 4)
        assert w1 == B.demons_workspace_bytes(ctx, 2) and w4 > 3 * (w1 - 5 * 4 * 16 * 12 * 10)
        assert B.demons_workspace_bytes_batch(ctx, 2, 0) == 0 and B.demons_workspace_bytes_batch(ctx, 2, 65) == 0
        vol = np.zeros((4, 10, 12, 16), np.float32)
        fld = np.zeros((4, 3, 10, 12, 16), np.float32)
        for nb in (0, 65):
            with pytest.raises(B.DemonsError) as e:
                B.demons_register_batch(ctx, nb, vol, vol, fld, None, [2, 2])
            assert e.value.code == B.E_ARG
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_batch(ctx, 4, vol, vol, fld, fld, [2, 2])      # u_back for a non-IC variant
        assert e.value.code == B.E_ARG
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_batch(ctx, 4, vol, vol, fld, None, [2, 2])     # valid arguments, but no workspace / device
        assert e.value.code == B.E_WORKSPACE
        slab = np.zeros((3, 6, 12, 16), np.float32)
        bad = [dict(z_begin=-1), dict(z_begin=6, z_count=6), dict(z_count=1), dict(own_begin=5, own_count=3), dict(own_count=-1)]
        for kw in bad:
            a = dict(z_begin=2, z_count=6, own_begin=1, own_count=4)
            a.update(kw)
            with pytest.raises(B.DemonsError) as e:
                B.demons_warp_force_slab(ctx, dims, a["z_begin"], a["z_count"], a["own_begin"], a["own_count"], vol[0], vol[0],
                                         slab, slab.copy())
            assert e.value.code == B.E_ARG, kw
        with pytest.raises(B.DemonsError) as e:
            B.demons_warp_force_slab(ctx, dims, 2, 6, 1, 4, vol[0], vol[0], slab, slab)   # aliased output
        assert e.value.code == B.E_ARG
    finally:
        B.demons_destroy(ctx)


def test_host_queue_arguments_validated(B):
    """Host-side validation of demons_register_host_queue (no device needed): the queue workspace is the single
    registration's plus one more staging slot (2 N floats of images, 3 N of field)."""
    import numpy as np
    dims = (16, 12, 10)
    n_vox = 16 * 12 * 10
    ctx = B.demons_create(dims, (1.0, 1.0, 1.0), B.PASSIVE, 1.0, 1.0)
    try:
        w1, wq = B.demons_workspace_bytes(ctx, 2), B.demons_workspace_bytes_queue(ctx, 2)
        assert 5 * 4 * n_vox <= wq - w1 <= 5 * 4 * n_vox + 3 * 256
        assert B.demons_workspace_bytes_queue(ctx, 0) == 0
        vol = np.zeros((10, 12, 16), np.float32)
        fld = np.zeros((3, 10, 12, 16), np.float32)
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_host_queue(ctx, [], [], [], None, [2, 2])               # empty queue
        assert e.value.code == B.E_ARG
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_host_queue(ctx, [vol], [vol], [fld], [fld], [2, 2])     # u_back for a non-IC variant
        assert e.value.code == B.E_ARG
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_host_queue(ctx, [vol, vol], [vol, vol], [fld, fld], None, [2, -1])
        assert e.value.code == B.E_ARG
        with pytest.raises(B.DemonsError) as e:
            B.demons_register_host_queue(ctx, [vol, vol], [vol, vol], [fld, fld], None, [2, 2])   # no workspace
        assert e.value.code == B.E_WORKSPACE
    finally:
        B.demons_destroy(ctx)
