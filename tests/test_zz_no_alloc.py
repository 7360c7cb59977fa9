"""nhp_soft_from_hard_noalloc against the existing path (nhp_render_obstacles_dt).

Who the entry point is for: code that must not allocate device memory once it is running -- a planner inside a control loop
with a fixed, audited memory budget, where cudaMalloc's driver lock and device-wide wait have no latency bound, or a guest in
a process whose framework already owns almost all of HBM, where cudaMalloc just fails.  Such a caller cannot create a planner
handle (nhp_planner_create allocates), so this call takes none: its scratch image is an array built into the library.

What is checked: the soft image and the distances are the ones the handle-based path produces, bit for bit (the tolerance the
distance-transform parity test uses), on two calls in a row and a third -- sizes going down and up again, so the second call
finds the first call's larger image still in the shared scratch and the third finds both; that free device memory does not move
across the calls; that a size beyond the built-in array is refused with a message naming the limit.

The file sorts after every other test file on purpose: `pytest -x` stops at the first failure and this entry point is an extra,
so a failure here must not hide the parity tests.  It passes alone in a fresh process (it then performs the per-device set-up
itself) and after the other tests."""
import numpy as np
import pytest

import scenes

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nhp():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2306_01301_b200 as nhp
    nhp.load_library()
    return nhp


def existing_path(nhp, sc, k):
    """soft image (uint8) and distances (float32) from the handle-based path, as numpy arrays"""
    import torch
    p = nhp.Planner.from_scene(sc)
    dist = torch.empty((sc.n, sc.n), dtype=torch.float32, device=p.device)
    p.render_obstacles_dt(sc.hard, k, dist)
    out = p.soft_image_numpy(), dist.cpu().numpy()
    p.close()
    return out


def test_two_calls_in_a_row_match_the_existing_path(nhp):
    import torch
    dev = torch.device("cuda:0")
    cases = [(scenes.random_scene(8, 5, 4.5, 31, vehicle=(3, 2), n_rects=40, soft=True), 4.0),     # 256 x 256
             (scenes.random_scene(6, 6, 8, 32, n_rects=9, soft=True), 11.5),                        # 64 x 64: a corner of the scratch the first call filled
             (scenes.get_config(4), 4.0)]                                                            # 512 x 512 (the soft benchmark scene)
    want = [existing_path(nhp, sc, k) for sc, k in cases]
    # every buffer is the caller's and exists before the first call
    hard = [torch.from_numpy(sc.hard).to(dev) for sc, _ in cases]
    soft = [torch.full((sc.n, sc.n), 7, dtype=torch.uint8, device=dev) for sc, _ in cases]
    dist = [torch.full((sc.n, sc.n), -1.0, dtype=torch.float32, device=dev) for sc, _ in cases]
    host_soft = [torch.empty((sc.n, sc.n), dtype=torch.uint8).pin_memory() for sc, _ in cases]
    host_dist = [torch.empty((sc.n, sc.n), dtype=torch.float32).pin_memory() for sc, _ in cases]
    torch.cuda.synchronize()

    def run_all():
        for c, (sc, k) in enumerate(cases):                     # back to back on one stream: no host wait in between
            nhp.soft_from_hard_noalloc(hard[c], k, soft[c], dist[c])
        for c in range(len(cases)):
            host_soft[c].copy_(soft[c], non_blocking=True)
            host_dist[c].copy_(dist[c], non_blocking=True)
        torch.cuda.synchronize()
        for c, (sc, k) in enumerate(cases):
            assert (host_soft[c].numpy() == want[c][0]).all(), (sc.name, "soft")
            assert (host_dist[c].numpy() == want[c][1]).all(), (sc.name, "dist")

    run_all()                                                   # includes the first call on this device (its set-up)
    for c in range(len(cases)):
        soft[c].fill_(0)
        dist[c].fill_(-2.0)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    run_all()
    run_all()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)                       # nothing was allocated or freed on the device
    # the distances are optional
    s2 = torch.zeros_like(soft[1])
    nhp.soft_from_hard_noalloc(hard[1], cases[1][1], s2)
    assert (s2.cpu().numpy() == want[1][0]).all()


def test_any_size_up_to_the_limit_and_none_beyond(nhp):
    import torch
    dev = torch.device("cuda:0")
    # a size the handle-based path does not offer (not a power of two): check against the definition on a few pixels' worth of
    # brute force done here in numpy -- exact squared distance to the nearest pixel of hard | row 0 | column 0
    n = 100
    rng = np.random.Generator(np.random.PCG64(5))
    h = (rng.random((n, n)) < 0.01).astype(np.uint8)
    hard = torch.from_numpy(h).to(dev)
    soft = torch.zeros((n, n), dtype=torch.uint8, device=dev)
    dist = torch.zeros((n, n), dtype=torch.float32, device=dev)
    nhp.soft_from_hard_noalloc(hard, 4.0, soft, dist)
    H = h.copy()
    H[0, :] = 1
    H[:, 0] = 1
    ys, xs = np.nonzero(H)
    yy, xx = np.mgrid[0:n, 0:n]
    d2 = ((yy[..., None] - ys) ** 2 + (xx[..., None] - xs) ** 2).min(axis=-1)
    d = np.sqrt(d2.astype(np.float32))
    assert (dist.cpu().numpy() == d).all()
    want = np.clip(np.rint(np.float32(16) * (np.float32(1) + np.float32(4) / (d + np.float32(1)))), 16, 255).astype(np.uint8)
    assert (soft.cpu().numpy() == want).all()
    # the largest size is accepted ...
    n = nhp.NOALLOC_MAX_N
    big = torch.zeros((n, n), dtype=torch.uint8, device=dev)
    out = torch.zeros((n, n), dtype=torch.uint8, device=dev)
    nhp.soft_from_hard_noalloc(big, 4.0, out)
    torch.cuda.synchronize()
    assert int(out[n - 1, n - 1]) == 16 and int(out[1, 1]) == 48          # far from the wall: 16 (1 + 4 / n) rounds to 16; next to it: 16 (1 + 4 / 2)
    # ... and the next one is refused with the limit in the message, before anything is launched
    n = nhp.NOALLOC_MAX_N + 1
    big = torch.zeros((n, n), dtype=torch.uint8, device=dev)
    out = torch.full((n, n), 9, dtype=torch.uint8, device=dev)
    with pytest.raises(nhp.NhpError) as e:
        nhp.soft_from_hard_noalloc(big, 4.0, out)
    assert e.value.code == -6 and str(nhp.NOALLOC_MAX_N) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 9).all())
    # host memory is not accepted
    L = nhp.load_library()
    host = np.zeros((64, 64), np.uint8)
    assert L.nhp_soft_from_hard_noalloc(host.ctypes.data, 64, 4.0, host.ctypes.data, None, None) == -6
    assert b"device memory" in L.nhp_noalloc_last_error()
