"""Parity of the Fourier-form (Eq.(7)-(9)) and shifted (Eq.(10)-(14)) Fresnel diffraction of the CUDA path against the
fp64 oracle, element by element.  Same bar as tests/test_gpu_parity.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_parity import REL_L2, MAX_ABS, _assert_parity, _dev, _rand, api   # noqa: E402,F401

LAM = 532e-9


def _gpu_fourier(api, u1, px, py, lam, z, inplace=False):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, px, lam)
    if px != py:
        plan.set_pitch_xy(px, py)
    d1 = _dev(u1)
    d2 = d1 if inplace else torch.empty_like(d1)
    api.cwo_fresnel_fourier(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


def _gpu_shifted(api, u1, p0, p1, lam, z, off=(0.0, 0.0), inplace=False):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, p0[0], lam)
    if p0[0] != p0[1]:
        plan.set_pitch_xy(*p0)
    if p1 is not None:
        plan.set_dst_pitch_xy(*p1)
    plan.set_offset(*off)
    d1 = _dev(u1)
    d2 = d1 if inplace else torch.empty_like(d1)
    api.cwo_fresnel_shifted(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


@pytest.mark.parametrize("shape", [(256, 256), (512, 256), (256, 1024), (1024, 1024), (2048, 512), (256, 4096),
                                   (8192, 256), (2048, 2048)])
def test_fourier_form_sizes_both_directions(api, oracle, shape):
    # every lane-pair tile shape (16, 8, 4, 2 lines per tile), the radix-2/4/8 leading stages, Nx != Ny, px != py, z < 0
    u1 = _rand(shape, 90 + shape[1] % 11)
    px, py = 6e-6, 9e-6
    for z in (0.05, -0.08):
        _assert_parity(_gpu_fourier(api, u1, px, py, LAM, z), oracle.fresnel_fourier(u1, px, py, LAM, z),
                       "fourier %s z=%g" % (shape, z))


def test_fourier_form_inplace_and_delta(api, oracle):
    u1 = _rand((512, 512), 97)
    ref = oracle.fresnel_fourier(u1, 8e-6, 8e-6, LAM, 0.1)
    _assert_parity(_gpu_fourier(api, u1, 8e-6, 8e-6, LAM, 0.1, inplace=True), ref, "fourier in place")
    # a single sample away from the centre: the result is a pure chirp with the coefficient's modulus everywhere
    d = np.zeros((256, 512), np.complex64); d[40, 300] = 1
    got = _gpu_fourier(api, d, 8e-6, 5e-6, LAM, 0.02)
    _assert_parity(got, oracle.fresnel_fourier(d, 8e-6, 5e-6, LAM, 0.02), "fourier delta")
    assert np.allclose(np.abs(got), 8e-6 * 5e-6 / (LAM * 0.02), rtol=1e-5)


def test_fourier_form_4096_sampled_against_the_direct_sum(api, oracle):
    # full size of the fresnel4096 workloads; 48 outputs against the direct sum of Eq.(1) at the destination pitch
    n, p, z = 4096, 4e-6, 0.5
    u1 = _rand((n, n), 98)
    got = _gpu_fourier(api, u1, p, p, LAM, z)
    r = np.random.default_rng(3)
    ms = np.concatenate([[0, n - 1, 0, n - 1, n // 2], r.integers(0, n, 43)])
    ns = np.concatenate([[0, n - 1, n - 1, 0, n // 2], r.integers(0, n, 43)])
    p2 = LAM * z / (n * p)
    oracle.set_threads(oracle.max_threads())
    ref = oracle.fresnel_general_points(u1, (p, p), (p2, p2), LAM, z, ms, ns)
    oracle.set_threads(min(8, oracle.max_threads()))
    err = np.abs(got[ns, ms] - ref)
    assert np.linalg.norm(err) / np.linalg.norm(ref) <= REL_L2 and err.max() <= MAX_ABS * np.abs(ref).max()


@pytest.mark.parametrize("shape", [(256, 256), (256, 512), (1024, 256), (1024, 1024), (512, 2048), (4096, 256),
                                   (256, 8192), (2048, 2048)])
def test_shifted_fresnel_pitch_and_offset(api, oracle, shape):
    u1 = _rand(shape, 120 + shape[0] % 13)
    p0, p1, off = (8e-6, 6e-6), (5e-6, 9e-6), (-310e-6, 170e-6)
    for z in (0.2, -0.15):
        _assert_parity(_gpu_shifted(api, u1, p0, p1, LAM, z, off), oracle.fresnel_shifted(u1, p0, p1, LAM, z, o1=off),
                       "shifted %s z=%g" % (shape, z))


def test_shifted_fresnel_special_cases(api, oracle):
    u1 = _rand((512, 1024), 131)
    p0 = (8e-6, 8e-6)
    # default destination grid: the convolution form
    _assert_parity(_gpu_shifted(api, u1, p0, None, LAM, 0.1), oracle.fresnel_conv(u1, 8e-6, 8e-6, LAM, 0.1), "shifted == conv")
    # magnification only, offset only, in place
    _assert_parity(_gpu_shifted(api, u1, p0, (16e-6, 4e-6), LAM, 0.1), oracle.fresnel_shifted(u1, p0, (16e-6, 4e-6), LAM, 0.1),
                   "shifted, pitch only")
    ref = oracle.fresnel_shifted(u1, p0, p0, LAM, 0.1, o1=(1.2e-3, -0.7e-3))
    _assert_parity(_gpu_shifted(api, u1, p0, p0, LAM, 0.1, (1.2e-3, -0.7e-3)), ref, "shifted, offset only")
    _assert_parity(_gpu_shifted(api, u1, p0, p0, LAM, 0.1, (1.2e-3, -0.7e-3), inplace=True), ref, "shifted in place")
    # the Fourier form's grid reached by the scaled convolution
    n = 512
    v = _rand((n, n), 132)
    p2 = LAM * 0.1 / (n * 8e-6)
    _assert_parity(_gpu_shifted(api, v, p0, (p2, p2), LAM, 0.1), oracle.fresnel_fourier(v, 8e-6, 8e-6, LAM, 0.1),
                   "shifted at the Fourier pitch")


def test_shifted_and_fourier_error_codes(api):
    plan = api.cwo_plan(128, 256, 8e-6, LAM)             # 128 < 256: outside the range of these two calls
    u = torch.zeros((256, 128), dtype=torch.complex64, device="cuda")
    for call in (api.cwo_fresnel_fourier, api.cwo_fresnel_shifted):
        with pytest.raises(api.CwoError) as e:
            call(plan, u, u, 0.1)
        assert e.value.code == api.CWO_EINVAL
    plan = api.cwo_plan(256, 256, 8e-6, LAM)
    u = torch.zeros((256, 256), dtype=torch.complex64, device="cuda")
    for call in (api.cwo_fresnel_fourier, api.cwo_fresnel_shifted):
        with pytest.raises(api.CwoError) as e:
            call(plan, u, u, 0.0)
        assert e.value.code == api.CWO_EINVAL
    with pytest.raises(api.CwoError):
        plan.set_dst_pitch_xy(5e-6, 0.0)


# ---- both ways of switching axes in the separable form (include/cwo_debug.h cwo_debug_set_fresnel_gather) ----------

@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("shape", [(256, 256), (512, 2048), (2048, 1024), (8192, 256), (256, 8192), (4096, 1024)])
def test_fresnel_conv_transposing_and_gathering_forms(api, oracle, mode, shape):
    # the default picks one of the two by field size; here each is forced on every tile shape, incl. the persistent
    # 8192-point kernel with its gathered prefetch, Nx != Ny, px != py, both signs of z, in place
    from paper_1107_5578_b200 import workloads as W
    cfg = W.CONFIGS["c5"]
    ny, nx = shape
    u1 = _rand(shape, 140 + ny % 17)
    px, py = cfg.pitch, 1.3 * cfg.pitch
    plan = api.cwo_plan(nx, ny, px, cfg.lam)
    plan.set_pitch_xy(px, py)
    plan.set_fresnel_gather(mode)
    for z in (cfg.zs[0] * max(shape) / 8192, -0.11):
        d1 = _dev(u1); d2 = torch.empty_like(d1)
        api.cwo_fresnel_conv(plan, d1, d2, z)
        api.cwo_fresnel_conv(plan, d1, d1, z)
        torch.cuda.synchronize()
        ref = oracle.fresnel_conv(u1, px, py, cfg.lam, z)
        _assert_parity(d2.cpu().numpy(), ref, "fresnel mode %d %s z=%g" % (mode, shape, z))
        _assert_parity(d1.cpu().numpy(), ref, "fresnel in place mode %d %s z=%g" % (mode, shape, z))


@pytest.mark.parametrize("mode", [0, 1])
def test_shifted_and_gs_in_both_forms(api, oracle, mode):
    from paper_1107_5578_b200 import workloads as W
    from test_gpu_parity import _phasor_rel_l2
    # shifted Fresnel
    u1 = _rand((1024, 512), 151)
    p0, p1, off = (8e-6, 6e-6), (5e-6, 9e-6), (-310e-6, 170e-6)
    plan = api.cwo_plan(512, 1024, p0[0], LAM)
    plan.set_pitch_xy(*p0); plan.set_dst_pitch_xy(*p1); plan.set_offset(*off); plan.set_fresnel_gather(mode)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    api.cwo_fresnel_shifted(plan, d1, d2, 0.2)
    torch.cuda.synchronize()
    _assert_parity(d2.cpu().numpy(), oracle.fresnel_shifted(u1, p0, p1, LAM, 0.2, o1=off), "shifted mode %d" % mode)
    # Gerchberg-Saxton, Fresnel propagator: kinoform and two loop passes from the oracle's state (non-square: the
    # layouts [Ny][Nx] and [Nx][Ny] alternate)
    cfg = W.CONFIGS["c5"]
    shape = (512, 1024)
    z = cfg.zs[0] * 1024 / 8192
    amp_src, amp_dst, phi0 = W.gs_inputs(shape, 9)
    plan = api.cwo_plan(shape[1], shape[0], cfg.pitch, cfg.lam)
    plan.set_fresnel_gather(mode)
    for iters in (0, 2):
        ph = _dev(phi0.astype(np.float32))
        api.cwo_gs(plan, _dev(amp_src), _dev(amp_dst), z, iters, ph)
        torch.cuda.synchronize()
        p = oracle.gs_init(0, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z)
        for _ in range(iters):
            p = oracle.gs_iter(0, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z)
        val = _phasor_rel_l2(ph.cpu().numpy(), p)
        print("MEASURED gs 512x1024 mode %d iters %d: phasor rel-L2 %.3e" % (mode, iters, val))
        # measured on the B200: 1.1e-6 (kinoform), 5.9e-6 (two iterations): the propagation bar itself holds
        assert val <= REL_L2, "gs mode %d iters %d" % (mode, iters)


@pytest.mark.parametrize("seed", range(10))
def test_random_shapes_and_parameters_fourier_and_shifted(api, oracle, seed):
    # seeded sweep over shapes (both tile orders), pitches, wavelengths, distances, destination pitches and offsets
    r = np.random.default_rng(500 + seed)
    ny, nx = (int(2 ** r.integers(8, 12)), int(2 ** r.integers(8, 12)))
    lam = float(r.choice([405e-9, 532e-9, 633e-9]))
    px, py = float(r.uniform(3e-6, 12e-6)), float(r.uniform(3e-6, 12e-6))
    z = float(r.uniform(0.02, 0.6) * r.choice([-1.0, 1.0]))
    u1 = _rand((ny, nx), 600 + seed)
    _assert_parity(_gpu_fourier(api, u1, px, py, lam, z), oracle.fresnel_fourier(u1, px, py, lam, z),
                   "fourier %dx%d z=%g" % (ny, nx, z))
    p1 = (float(px * r.uniform(0.5, 2.0)), float(py * r.uniform(0.5, 2.0)))
    off = (float(r.uniform(-1, 1) * nx * px), float(r.uniform(-1, 1) * ny * py))
    _assert_parity(_gpu_shifted(api, u1, (px, py), p1, lam, z, off), oracle.fresnel_shifted(u1, (px, py), p1, lam, z, o1=off),
                   "shifted %dx%d z=%g" % (ny, nx, z))
