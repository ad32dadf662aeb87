"""fdgs_render_forward_static (include/fdgs.h): the forward of one view on the workspace that is built into the library
as a device array, for callers that cannot allocate.  It must give what the existing path gives — fdgs_preprocess +
fdgs_render_forward on a caller-owned workspace — on two calls in a row (the second starts from what the first left in
the shared array), must not take device memory, and must refuse sizes beyond its limit.

Collected last on purpose (the suite runs with pytest -x)."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2412_20720_b200 import scenes

N, WIDTH, HEIGHT, CAP = 30000, 320, 240, 393216


def _workspace_path(fdgs, ds, view):
    """The existing path: caller-owned workspace (torch allocation), fdgs_preprocess + fdgs_render_forward."""
    import torch
    r = fdgs.Renderer(ds, view.width, view.height, CAP)
    cv = fdgs.make_view(view)
    D, nvis = r.preprocess(cv, sync=True)
    r.forward(cv)
    torch.cuda.synchronize()
    return D, nvis, r.image.cpu().numpy(), r.final_T.cpu().numpy(), r.n_contrib.cpu().numpy()


def test_static_forward_equals_the_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=N, width=WIDTH, height=HEIGHT, n_views=2)
    ds = fdgs.DeviceScene.from_scene(sc)
    assert fdgs.workspace_bytes(ds.N, ds.K, WIDTH, HEIGHT, CAP) <= fdgs.STATIC_WS_BYTES
    dev = ds.mean.device
    image = torch.empty((3, HEIGHT, WIDTH), dtype=torch.float32, device=dev)
    final_T = torch.empty((HEIGHT, WIDTH), dtype=torch.float32, device=dev)
    n_contrib = torch.empty((HEIGHT, WIDTH), dtype=torch.int32, device=dev)
    overflow = torch.empty(1, dtype=torch.int32, device=dev)
    expected = [_workspace_path(fdgs, ds, v) for v in sc.views[:2]]
    # several tiles of the depth sort (2048 keys) and several chunks of the row scatter (2048 survivors)
    assert expected[0][0] > 15000 and expected[0][1] > 4096, f"scene too small: D = {expected[0][0]}, visible = {expected[0][1]}"
    assert not np.array_equal(expected[0][2], expected[1][2]), "the two views must differ (camera and time)"
    for call, (view, (D, nvis, img_e, T_e, nc_e)) in enumerate(zip(sc.views[:2], expected)):
        image.fill_(float("nan")); final_T.fill_(float("nan")); n_contrib.fill_(-1); overflow.fill_(-1)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        fdgs.render_forward_static(ds, fdgs.make_view(view), CAP, image, final_T, n_contrib, overflow)
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info()[0]
        if call == 1:       # the first call of a process may load kernels (module memory); the second takes nothing
            assert free_after == free_before, f"device memory changed by {free_before - free_after} bytes"
        assert int(overflow.item()) == 0
        # same kernels on the same inputs: the tolerance of this comparison is zero
        assert np.array_equal(n_contrib.cpu().numpy(), nc_e), f"call {call}: n_contrib differs"
        assert np.array_equal(final_T.cpu().numpy(), T_e), f"call {call}: final_T differs"
        got = image.cpu().numpy()
        assert np.isfinite(got).all()
        assert np.array_equal(got, img_e), f"call {call}: image differs, max abs {np.abs(got - img_e).max()}"


def test_static_forward_reports_pair_overflow_on_the_device():
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=N, width=WIDTH, height=HEIGHT, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    dev = ds.mean.device
    image = torch.empty((3, HEIGHT, WIDTH), dtype=torch.float32, device=dev)
    final_T = torch.empty((HEIGHT, WIDTH), dtype=torch.float32, device=dev)
    n_contrib = torch.empty((HEIGHT, WIDTH), dtype=torch.int32, device=dev)
    overflow = torch.zeros(1, dtype=torch.int32, device=dev)
    fdgs.render_forward_static(ds, fdgs.make_view(sc.views[0]), 1000, image, final_T, n_contrib, overflow)
    torch.cuda.synchronize()
    assert int(overflow.item()) == 1
    assert (n_contrib == 0).all() and (final_T == 1).all()      # nothing drawn: the image of an empty rendering


def test_static_forward_refuses_sizes_beyond_its_workspace():
    import torch
    from paper_2412_20720_b200 import fdgs
    sc = scenes.multiview_video(N=2000, width=WIDTH, height=HEIGHT, n_views=1)
    ds = fdgs.DeviceScene.from_scene(sc)
    dev = ds.mean.device
    image = torch.full((3, HEIGHT, WIDTH), 7.0, dtype=torch.float32, device=dev)
    final_T = torch.empty((HEIGHT, WIDTH), dtype=torch.float32, device=dev)
    n_contrib = torch.empty((HEIGHT, WIDTH), dtype=torch.int32, device=dev)
    cap_too_large = 4 << 20                                     # 16 MiB of ids alone
    assert fdgs.workspace_bytes(ds.N, ds.K, WIDTH, HEIGHT, cap_too_large) > fdgs.STATIC_WS_BYTES
    launches = fdgs.load().fdgs_launch_count()
    with pytest.raises(fdgs.FdgsError) as e:
        fdgs.render_forward_static(ds, fdgs.make_view(sc.views[0]), cap_too_large, image, final_T, n_contrib)
    assert e.value.code == fdgs.ERR_STATIC_LIMIT and "FDGS_STATIC_WS_BYTES" in str(e.value)
    torch.cuda.synchronize()
    assert fdgs.load().fdgs_launch_count() == launches and (image == 7.0).all()     # nothing was launched
    # one million primitives do not fit either, whatever the pointers are: the size check comes first
    big = fdgs.CScene(1_000_000, 3, 1, None, None, None, None, None, None)
    cfg = fdgs.default_config()
    rc = fdgs.load().fdgs_render_forward_static(C.byref(big), C.byref(fdgs.make_view(sc.views[0])), C.byref(cfg), 65536, None,
                                                image.data_ptr(), final_T.data_ptr(), n_contrib.data_ptr(), None)
    assert rc == fdgs.ERR_STATIC_LIMIT
    # and a size that fits still renders afterwards
    fdgs.render_forward_static(ds, fdgs.make_view(sc.views[0]), 65536, image, final_T, n_contrib)
    torch.cuda.synchronize()
    assert torch.isfinite(image).all() and not (image == 7.0).all()
