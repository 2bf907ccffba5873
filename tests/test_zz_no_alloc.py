"""aepid_gamma_of_upsampled_static (include/aepid.h): the one entry point that allocates nothing (no context, no workspace; its
scratch is a file-scope static device array of the library, AEPID_STATIC_MAX_PIXELS floats + 256 bytes).  Its output is checked
against the existing path (aepid_upsample + aepid_gamma_index on a context with a caller workspace), on two calls in a row with
different images, grids and criteria (the array keeps the first call's contents), within the tolerance the analysis tests use
(tests/test_gpu_analysis.py: 3e-5 absolute on gamma; the kernels are the same, so the maps come out identical).
This file is collected last on purpose: the suite runs with pytest -x."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

GAMMA_TOL = 3e-5          # DESIGN.md section 7, K10


def image(nv, nu, seed, noise=0.0):
    """Smooth IMRT-like image: soft-edged rectangles on a low background (inputs only, no method arithmetic)."""
    rng = np.random.default_rng(seed)
    y, x = np.mgrid[0:nv, 0:nu].astype(np.float64)
    img = np.full((nv, nu), 0.02)
    for _ in range(5):
        cx, cy = rng.uniform(0.3, 0.7) * nu, rng.uniform(0.3, 0.7) * nv
        wx, wy = rng.uniform(0.08, 0.25) * nu, rng.uniform(0.08, 0.25) * nv
        edge = 0.015 * nu
        img += rng.uniform(0.2, 1.0) / ((1 + np.exp((np.abs(x - cx) - wx) / edge)) * (1 + np.exp((np.abs(y - cy) - wy) / edge)))
    if noise:
        img *= 1 + noise * rng.standard_normal(img.shape)
    return np.maximum(img, 0.0).astype(np.float32)


def test_static_scratch_entry_point_matches_the_context_path_on_two_calls_in_a_row():
    import torch
    from gen import make_config
    from paper_2510_24154_b200 import AepidError, Engine, gamma_of_upsampled_static
    from paper_2510_24154_b200.binding import STATIC_MAX_PIXELS
    dev = torch.device("cuda", 0)
    # (predicted grid, measured grid, pitch of the measured grid in cm, dose criterion, DTA in cm): the paper's chain
    # 160 x 160 -> 1190 x 1190 at 3 %/3 mm, then a smaller, non-square case at 2 %/2 mm
    cases = [((160, 160), (1190, 1190), 40.0 / 1190, 0.03, 0.3, 33), ((96, 128), (500, 620), 0.06, 0.02, 0.2, 34)]
    inputs = []
    for (nv, nu), (mv, mu), pitch, frac, dta, seed in cases:
        pred = torch.from_numpy(image(nv, nu, seed)).to(dev)
        meas = torch.from_numpy(image(mv, mu, seed, noise=0.02)).to(dev)
        inputs.append((pred, meas, pitch, frac, dta))

    # the existing path: a context with a caller-provided workspace
    cfg = make_config("C0")
    eng = Engine.for_config(cfg); eng.load_config(cfg)
    want = []
    for pred, meas, pitch, frac, dta in inputs:
        up = eng.upsample(pred, meas.shape[0], meas.shape[1])
        g, st = eng.gamma_index(meas, up, pitch, frac, dta, 0.10, 2.0)
        want.append((g.cpu().numpy(), st))
    eng.close()

    # the new entry point: outputs are the caller's, made before the calls; one call first (it resolves the address of the
    # static array on this device), then the two calls in a row that are checked, with the free device memory watched
    outs = [(torch.empty_like(m), torch.empty(4, dtype=torch.float64, device=dev)) for _, m, _, _, _ in inputs]
    warm = (torch.empty_like(inputs[1][1]), torch.empty(4, dtype=torch.float64, device=dev))
    p, m, pitch, frac, dta = inputs[1]
    gamma_of_upsampled_static(p, m, pitch, frac, dta, 0.10, 2.0, out=warm[0], stats_out=warm[1])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info(dev)[0]
    for (pred, meas, pitch, frac, dta), (g, s) in zip(inputs, outs):
        gamma_of_upsampled_static(pred, meas, pitch, frac, dta, 0.10, 2.0, out=g, stats_out=s)      # back to back, same stream
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info(dev)[0]
    assert free0 - free1 < (1 << 20), "the calls took %d bytes of device memory" % (free0 - free1)

    for (g, s), (gw, stw), (pred, meas, pitch, frac, dta) in zip(outs, want, inputs):
        gg, ss = g.cpu().numpy(), s.cpu().numpy()
        assert np.array_equal(gg < 0, gw < 0)                              # the same pixels are tested
        assert np.abs(gg - gw).max() <= GAMMA_TOL
        assert ss[0] == stw["n_tested"] and ss[0] > 10000 and ss[1] == stw["n_pass"]
        assert abs(ss[2] - stw["mean_gamma"]) <= GAMMA_TOL and abs(ss[3] - stw["max_gamma"]) <= GAMMA_TOL
        print("static entry point: %d x %d -> %d x %d, %d pixels tested, pass rate %.4f, max |gamma - context path| = %.1e"
              % (pred.shape[0], pred.shape[1], meas.shape[0], meas.shape[1], ss[0], ss[1] / ss[0], np.abs(gg - gw).max()))
    # the warm-up call computed the second case as well
    assert np.abs(warm[0].cpu().numpy() - want[1][0]).max() <= GAMMA_TOL

    # limits and errors: a measured grid beyond the static maximum is refused with a message that says so; host memory is refused
    n = int(np.sqrt(STATIC_MAX_PIXELS)) + 1
    big = torch.zeros((n, n), dtype=torch.float32, device=dev)
    with pytest.raises(AepidError, match="NOMEM.*AEPID_STATIC_MAX_PIXELS"):
        gamma_of_upsampled_static(inputs[0][0], big, 0.03, out=big.clone())
    edge = torch.ones((1280, 1280), dtype=torch.float32, device=dev)      # exactly the maximum is accepted
    gamma_of_upsampled_static(inputs[0][0], edge, 0.03, out=torch.empty_like(edge))
    torch.cuda.synchronize()
    with pytest.raises(AepidError, match="BAD_ARG"):
        gamma_of_upsampled_static(inputs[0][0], inputs[0][1], -1.0)
    with pytest.raises(AepidError, match="NOMEM.*shared memory"):
        gamma_of_upsampled_static(inputs[0][0], inputs[0][1], 0.002, 0.03, 0.3)      # a search window of 300 pixels
    # raw C-ABI call with HOST images: refused, not dereferenced on the device
    import ctypes as C
    from paper_2510_24154_b200 import load_library
    lib = load_library()
    h = np.ones((64, 64), dtype=np.float32); ho = np.empty((64, 64), dtype=np.float32)
    err = C.create_string_buffer(256)
    rc = lib.aepid_gamma_of_upsampled_static(0, None, h.ctypes.data_as(C.c_void_p), 64, 64, h.ctypes.data_as(C.c_void_p), 64, 64,
                                             C.c_float(0.1), C.c_float(0.03), C.c_float(0.3), C.c_float(0.1), C.c_float(2.0),
                                             ho.ctypes.data_as(C.c_void_p), None, err, len(err))
    assert rc == -1 and b"device pointers" in err.value
