"""blink_image_static: imaging for callers that cannot allocate device memory.

blink_image needs plan scratch, and plan scratch comes from blink_plan_reserve = cudaMalloc.  A real-time
loop behind a correlator cannot take that call's device-wide stall, and a process whose GPU memory is
already owned by something else cannot count on it succeeding; blink_image_static gives them the same
images with the intermediate held in a 32 MiB array compiled into libblink.so (include/blink.h).

What is checked here: its images against blink_image's on the same grids -- bit for bit where blink_image
itself runs the line kernels, within the image bar of the parity tests (1e-4 of the peak) where blink_image
takes another route -- on TWO calls in a row with different data, grid size and batch shape, so that
whatever the first call left in the shared array would show up in the second; that the plan it ran on
never acquired scratch; that a repeat call leaves the device's free memory where it was; and that a plan
whose single snapshot does not fit the array is turned away with BLINK_ECAPACITY before anything runs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure of this
add-on must not hide the parity tests.  It holds no state from other tests and passes alone in a fresh
process as well as after them.
"""
import numpy as np
import pytest

from paper_2405_13478_b200 import synth

pytestmark = pytest.mark.gpu

IMG_TOL = 1e-4     # the image bar of tests/test_gpu_parity.py


def _case(name):
    if name == "station128":      # blink_image = line kernels: bit-identical expected; one launch pair
        return synth.config_station(n_t=2, n_ch=3, n_pix=128), True
    if name == "mwa1":            # blink_image = residue-class kernel; 12 snapshots of 4 MiB = 2 launch pairs
        return synth.config_mwa1(n_t=4, n_ch=3), False
    if name == "station_uniform_32":
        w = synth.config_station(n_t=3, n_ch=2, n_pix=32)
        w.weighting = synth.UNIFORM
        return w, True
    raise KeyError(name)


def _both_paths(torch, blink, name, seed_shift):
    """grids of one workload -> (images of blink_image_static, images of blink_image, bit-identical expected,
    the plan the static call ran on)"""
    w, same_kernels = _case(name)
    w.seed += seed_shift                       # other noise than the previous call's
    vis = torch.from_numpy(w.vis()).cuda()
    plan_s = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)   # never reserved
    plan_e = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)   # the existing path
    uv = plan_e.grid(vis)
    shape = (w.n_t, w.n_ch, w.n_pix, w.n_pix)
    img_s = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")      # must be fully overwritten
    img_e = torch.full(shape, float("nan"), dtype=torch.float32, device="cuda")
    plan_e.image(uv, img_e)                    # reserves plan scratch (cudaMalloc) -- what the other call avoids
    plan_s.image_static(uv, img_s)
    torch.cuda.synchronize()
    assert plan_s.query_i64(blink.Q_SCRATCH_BYTES) == 0, "blink_image_static must not acquire plan scratch"
    plan_e.close()
    return img_s, img_e, same_kernels, plan_s, uv


def _compare(img_s, img_e, same_kernels, what):
    a, b = img_s.cpu().numpy(), img_e.cpu().numpy()
    assert np.all(np.isfinite(a)), f"{what}: image not fully overwritten"
    if same_kernels:
        assert np.array_equal(a, b), f"{what}: same kernels, other scratch: images must be bit-identical"
    for s in range(a.shape[0] * a.shape[1]):
        x, y = a.reshape(-1, *a.shape[2:])[s], b.reshape(-1, *b.shape[2:])[s]
        peak = np.max(np.abs(y))
        err = np.max(np.abs(x - y))
        assert err <= IMG_TOL * peak, f"{what}, snapshot {s}: err {err:.3e} peak {peak:.3e}"


@pytest.mark.parametrize("first,second", [("station128", "mwa1"), ("mwa1", "station_uniform_32")])
def test_static_scratch_images_equal_blink_image_on_two_calls_in_a_row(torch_cuda, blink, first, second):
    torch = torch_cuda
    img_s, img_e, same, plan1, _ = _both_paths(torch, blink, first, 0)
    _compare(img_s, img_e, same, f"first call ({first})")
    plan1.close()
    # second call: other plan, other size, other data -- the array still holds the first call's intermediate
    img_s, img_e, same, plan2, uv = _both_paths(torch, blink, second, 17)
    _compare(img_s, img_e, same, f"second call ({second})")
    # a repeat of that call: same answer (bitwise), and the device's free memory does not move
    again = torch.full_like(img_s, float("nan"))
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    plan2.image_static(uv, again)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert torch.equal(again, img_s), "blink_image_static is not reproducible call to call"
    assert free_after == free_before, "device memory was allocated or freed during blink_image_static"
    plan2.close()


def test_static_scratch_against_oracle(torch_cuda, blink, oracle):
    """the same call against the CPU oracle (configs[0]), so that it does not rest on blink_image alone"""
    torch = torch_cuda
    w = synth.config_tiny()
    vis = w.vis()
    plan = blink.Plan(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting)
    uv = plan.grid(torch.from_numpy(vis).cuda())
    img = torch.full((w.n_t, w.n_ch, w.n_pix, w.n_pix), float("nan"), dtype=torch.float32, device="cuda")
    plan.image_static(uv, img)
    torch.cuda.synchronize()
    ref = oracle.image_batch(w.ant_enu_m, w.freq_hz, w.n_pix, w.pixscale, w.weighting, vis, np.array([0], np.int64))
    i_ref = ref["images"][0]
    err = np.max(np.abs(img.cpu().numpy()[0, 0] - i_ref))
    assert err <= IMG_TOL * np.max(np.abs(i_ref)), err
    plan.close()


def test_static_scratch_rejects_a_snapshot_that_does_not_fit(torch_cuda, blink):
    """N = 4096 with a half-plane wider than 1024 columns: 8 N wu > 32 MiB -> BLINK_ECAPACITY, a message
    with both numbers, nothing launched (the pointers are never dereferenced)."""
    torch = torch_cuda
    ant = np.array([[0.0, 0.0, 0.0], [1500.0, 0.0, 0.0], [0.0, 100.0, 0.0]])   # 750 wavelengths East at 150 MHz
    plan = blink.Plan(ant, np.array([150e6]), 4096, 2.0 / 4096, synth.NATURAL)
    kx_max, _ = plan.bbox(0)
    assert 8 * 4096 * (kx_max + 1) > blink.STATIC_SCRATCH_BYTES
    dummy_uv = torch.zeros(16, dtype=torch.complex64, device="cuda")
    dummy_img = torch.full((16,), float("nan"), dtype=torch.float32, device="cuda")
    lib = blink.load()
    rc = lib.blink_image_static(plan._h, dummy_uv.data_ptr(), 1, dummy_img.data_ptr(), None)
    assert rc == blink.ECAPACITY
    assert "built-in scratch" in lib.blink_strerror(rc).decode()
    msg = lib.blink_last_cuda_error().decode()
    assert str(blink.STATIC_SCRATCH_BYTES) in msg and "4096" in msg, msg
    torch.cuda.synchronize()
    assert bool(torch.isnan(dummy_img).all()), "a rejected call must not touch its outputs"
    # n_t = 0 stays a no-op, bad pointers stay BLINK_EINVAL
    assert lib.blink_image_static(plan._h, None, 0, None, None) == blink.OK
    assert lib.blink_image_static(plan._h, None, 1, dummy_img.data_ptr(), None) == blink.EINVAL
    plan.close()
