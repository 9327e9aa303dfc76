"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element.

Bar (BASELINE.json north_star): relative L2 <= 2e-5 and max abs error <= 1e-4 * peak |u2_oracle|,
fp32 against double on the same seeded complex64 inputs.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1107_5578_b200 import workloads as W   # noqa: E402

REL_L2, MAX_ABS = 2e-5, 1e-4


@pytest.fixture(scope="module")
def api():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1107_5578_b200 import api as a
    a.lib()
    return a


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _assert_parity(got, ref, what=""):
    got = np.asarray(got).astype(np.complex128); ref = np.asarray(ref)
    rel = np.linalg.norm((got - ref).ravel()) / np.linalg.norm(ref.ravel())
    mx = np.max(np.abs(got - ref)) / np.max(np.abs(ref))
    assert rel <= REL_L2 and mx <= MAX_ABS, "%s rel-L2 %.3e max/peak %.3e" % (what, rel, mx)
    return rel, mx


def _rand(shape, seed):
    r = np.random.default_rng(seed)
    return (r.standard_normal(shape) + 1j * r.standard_normal(shape)).astype(np.complex64)


def _gpu_asm(api, u1, px, py, lam, z, inplace=False):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, px, lam)
    if px != py:
        plan.set_pitch_xy(px, py)
    d1 = _dev(u1)
    d2 = d1 if inplace else torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


def _gpu_fresnel(api, u1, px, py, lam, z, inplace=False):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, px, lam)
    if px != py:
        plan.set_pitch_xy(px, py)
    d1 = _dev(u1)
    d2 = d1 if inplace else torch.empty_like(d1)
    api.cwo_fresnel_conv(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


# ---------------------------------------------------------------- ASM -----------------------------------------

@pytest.mark.parametrize("n", [32, 64, 128, 256, 512, 1024, 2048])
def test_asm_square_sizes(api, oracle, n):
    cfg = W.CONFIGS["c3"].scaled(n)
    u1 = W.make_field(cfg)
    for z in (0.01, -0.037):
        _assert_parity(_gpu_asm(api, u1, cfg.pitch, cfg.pitch, cfg.lam, z), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, z),
                       "asm %d z=%g" % (n, z))


@pytest.mark.parametrize("shape", [(32, 1024), (2048, 64), (256, 4096), (8192, 32), (32, 16384), (16384, 32),
                                   (1024, 4096), (4096, 1024), (2048, 1024), (1024, 8192), (8192, 2048)])
def test_asm_non_square_and_unequal_pitch(api, oracle, shape):
    u1 = _rand(shape, 3)
    px, py, lam, z = 3e-6, 5e-6, 633e-9, 0.004
    _assert_parity(_gpu_asm(api, u1, px, py, lam, z), oracle.asm(u1, px, py, lam, z), "asm %s" % (shape,))


def test_asm_c1_full(api, oracle):
    cfg = W.CONFIGS["c1"]
    u1 = W.make_field(cfg)
    _assert_parity(_gpu_asm(api, u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]),
                   oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]), "c1")


def test_asm_c3_full_all_distances(api, oracle):
    cfg = W.CONFIGS["c3"]
    u1 = W.make_field(cfg)
    plan = api.cwo_plan(cfg.N, cfg.N, cfg.pitch, cfg.lam)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    for z in cfg.zs:
        api.cwo_asm(plan, d1, d2, z)
        torch.cuda.synchronize()
        _assert_parity(d2.cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, z), "c3 z=%g" % z)


def test_asm_8192(api, oracle):
    u1 = W.make_field(W.CONFIGS["c3"].scaled(8192))
    _assert_parity(_gpu_asm(api, u1, 4e-6, 4e-6, 633e-9, 0.1), oracle.asm(u1, 4e-6, 4e-6, 633e-9, 0.1), "asm 8192")


def test_asm_z0_identity_inplace_and_roundtrip(api):
    u1 = _rand((512, 512), 5)
    out = _gpu_asm(api, u1, 4e-6, 4e-6, 633e-9, 0.0, inplace=True)
    _assert_parity(out, u1.astype(np.complex128), "z=0")
    fwd = _gpu_asm(api, u1, 4e-6, 4e-6, 633e-9, 0.02)
    back = _gpu_asm(api, fwd, 4e-6, 4e-6, 633e-9, -0.02)
    _assert_parity(back, u1.astype(np.complex128), "round trip")
    assert abs(np.linalg.norm(fwd.astype(np.complex128)) / np.linalg.norm(u1.astype(np.complex128)) - 1) < 1e-5


def test_asm_evanescent_classification(api, oracle):
    # pitch < lambda/sqrt(2): a large share of the bins is evanescent; one misclassified bin costs ~1/N
    n, d, lam = 64, 0.3e-6, 633e-9
    u1 = _rand((n, n), 7)
    for z in (5e-6, -5e-6):
        _assert_parity(_gpu_asm(api, u1, d, d, lam, z), oracle.asm(u1, d, d, lam, z), "evanescent z=%g" % z)
    jy, jx = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    pw = np.exp(2j * np.pi * (25 * jx + 20 * jy) / n).astype(np.complex64)      # f0 > 1/lambda
    assert np.max(np.abs(_gpu_asm(api, pw, d, d, lam, 5e-6))) < 1e-4


# ---------------------------------------------------------------- Fresnel ---------------------------------------

@pytest.mark.parametrize("n", [16, 32, 64, 128, 256, 512])
def test_fresnel_square_sizes(api, oracle, n):
    cfg = W.CONFIGS["c2"].scaled(n)
    u1 = _rand((n, n), n)
    z = cfg.zs[0] * n / 1024                      # keeps N pitch^2/(lambda z) as in c2
    for zz in (z, -z):
        _assert_parity(_gpu_fresnel(api, u1, cfg.pitch, cfg.pitch, cfg.lam, zz),
                       oracle.fresnel_conv(u1, cfg.pitch, cfg.pitch, cfg.lam, zz), "fresnel %d z=%g" % (n, zz))


@pytest.mark.parametrize("shape", [(16, 512), (1024, 32), (64, 2048), (512, 2048), (2048, 512), (1024, 4096), (4096, 1024)])
def test_fresnel_non_square_and_unequal_pitch(api, oracle, shape):
    u1 = _rand(shape, 11)
    px, py, lam, z = 6e-6, 9e-6, 532e-9, 0.01
    _assert_parity(_gpu_fresnel(api, u1, px, py, lam, z), oracle.fresnel_conv(u1, px, py, lam, z), "fresnel %s" % (shape,))


@pytest.mark.parametrize("shape", [(8192, 32), (32, 8192), (8192, 64), (64, 8192), (4096, 64), (64, 4096), (8192, 256)])
def test_fresnel_long_transforms_full_field(api, oracle, shape):
    """The 8192- and 16384-point transforms of c5 / Fresnel 8192^2, compared element by element: one axis at full
    length, the other short enough for the fp64 oracle (rows and columns both ways), at c5's pitch and wavelength."""
    cfg = W.CONFIGS["c5"]
    u1 = _rand(shape, 41 + shape[0] % 7)
    for z in (cfg.zs[0], -cfg.zs[0]):
        _assert_parity(_gpu_fresnel(api, u1, cfg.pitch, cfg.pitch, cfg.lam, z),
                       oracle.fresnel_conv(u1, cfg.pitch, cfg.pitch, cfg.lam, z), "fresnel %s z=%g" % (shape, z))


def test_fresnel_c2_full_and_inplace(api, oracle):
    cfg = W.CONFIGS["c2"]
    u1 = W.make_field(cfg)
    ref = oracle.fresnel_conv(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0])
    _assert_parity(_gpu_fresnel(api, u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]), ref, "c2")
    _assert_parity(_gpu_fresnel(api, u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0], inplace=True), ref, "c2 in place")


def test_fresnel_2048_and_4096(api, oracle):
    for n in (2048, 4096):
        u1 = W.make_field(W.CONFIGS["c2"].scaled(n))
        got = _gpu_fresnel(api, u1, 8e-6, 8e-6, 532e-9, 0.2 * n / 1024)
        if n == 2048:
            _assert_parity(got, oracle.fresnel_conv(u1, 8e-6, 8e-6, 532e-9, 0.2 * n / 1024), "fresnel 2048")
        else:
            # the whole field against the oracle's Eq.(5) pipeline (three fp64 FFTs of 8192^2) ...
            oracle.set_threads(oracle.max_threads())
            _assert_parity(got, oracle.fresnel_conv(u1, 8e-6, 8e-6, 532e-9, 0.2 * n / 1024), "fresnel 4096, full field")
            oracle.set_threads(min(8, oracle.max_threads()))
            # ... and sampled outputs against the direct sum of Eq.(1) per point (independent of the oracle's FFT)
            r = np.random.default_rng(1)
            ms = r.integers(0, n, 24); ns = r.integers(0, n, 24)
            ref = oracle.fresnel_points(u1, 8e-6, 8e-6, 532e-9, 0.2 * n / 1024, ms, ns)
            peak = np.abs(ref).max()
            err = np.abs(got[ns, ms] - ref)
            assert np.linalg.norm(err) / np.linalg.norm(ref) <= REL_L2 and err.max() <= MAX_ABS * peak


def test_fresnel_c5_size_sampled(api, oracle):
    # 8192^2 -> virtual 16384^2 in the launch configuration bench.py --workload c5 / fresnel8192 times: 256 outputs
    # against the direct sum of Eq.(1) (the oracle's plain definition), covering every row and column phase mod 8,
    # both crop edges and the corners; rel-L2 and max-abs gates as everywhere
    cfg = W.CONFIGS["c5"]
    n = cfg.N
    r = np.random.default_rng(2)
    u1 = W.random_phasor(cfg)
    got = _gpu_fresnel(api, u1, cfg.pitch, cfg.pitch, cfg.lam, -cfg.zs[0])
    edge = np.array([0, 1, 2, 3, n - 4, n - 3, n - 2, n - 1])
    ms = np.concatenate([[0, n - 1, 0, n - 1], edge, r.integers(0, n, 8), r.integers(0, n, 236)])
    ns = np.concatenate([[0, n - 1, n - 1, 0], r.integers(0, n, 8), edge, r.integers(0, n, 236)])
    ms[20:84] = (ms[20:84] // 8) * 8 + np.arange(64) % 8          # every x mod 8 ...
    ns[20:84] = (ns[20:84] // 8) * 8 + np.arange(64) // 8         # ... with every y mod 8
    assert ms.size == 256
    oracle.set_threads(oracle.max_threads())          # 256 direct sums over 8192^2 terms
    ref = oracle.fresnel_points(u1, cfg.pitch, cfg.pitch, cfg.lam, -cfg.zs[0], ms, ns)
    oracle.set_threads(min(8, oracle.max_threads()))
    err = np.abs(got[ns, ms] - ref)
    # the peak of |u2| is not known from samples: every |u1| is 1 and the operator is ~unitary, so the sample
    # maximum is a lower bound of the peak (a stricter gate than the definition's)
    assert np.linalg.norm(err) / np.linalg.norm(ref) <= REL_L2, (err.max(), np.abs(ref).max())
    assert err.max() <= MAX_ABS * np.abs(ref).max(), (err.max(), np.abs(ref).max())


# ---------------------------------------------------------------- stack ---------------------------------------

def test_stack_small_full(api, oracle):
    cfg = W.CONFIGS["c4"].scaled(256)
    u1 = W.make_field(cfg)
    zs = [0.001, 0.002, 0.0035, -0.001, 0.064]
    plan = api.cwo_plan(cfg.N, cfg.N, cfg.pitch, cfg.lam)
    out = torch.empty((len(zs), cfg.N, cfg.N), dtype=torch.complex64, device="cuda")
    api.cwo_propagate_stack(plan, _dev(u1), zs, out)
    torch.cuda.synchronize()
    ref = oracle.stack(u1, cfg.pitch, cfg.pitch, cfg.lam, zs)
    for k in range(len(zs)):
        _assert_parity(out[k].cpu().numpy(), ref[k], "stack plane %d" % k)


def test_stack_c4_full_size_sampled_planes(api, oracle):
    cfg = W.CONFIGS["c4"]
    u1 = W.make_field(cfg)
    plan = api.cwo_plan(cfg.N, cfg.N, cfg.pitch, cfg.lam)
    out = torch.empty((len(cfg.zs), cfg.N, cfg.N), dtype=torch.complex64, device="cuda")
    api.cwo_propagate_stack(plan, _dev(u1), cfg.zs, out)
    torch.cuda.synchronize()
    # every plane of the second 16-plane batch of launches (positions 0..15), and the first / last plane of the call
    for k in [0] + list(range(16, 32)) + [63]:
        _assert_parity(out[k].cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[k]), "c4 plane %d" % k)
    # every plane carries the input's energy (unitary H, no evanescent bins)
    e = torch.linalg.vector_norm(out.reshape(len(cfg.zs), -1), dim=1).cpu().numpy()
    assert np.allclose(e, np.linalg.norm(u1.astype(np.complex128)), rtol=1e-5)


# ---------------------------------------------------------------- GS ------------------------------------------

def _gs_gpu(api, method, amp_src, amp_dst, phi, pitch, lam, z, iters):
    ny, nx = amp_src.shape
    plan = api.cwo_plan(nx, ny, pitch, lam)
    plan.set_option(api.CWO_OPT_GS_METHOD, method)
    ph = _dev(phi.astype(np.float32))
    api.cwo_gs(plan, _dev(amp_src), _dev(amp_dst), z, iters, ph)
    torch.cuda.synchronize()
    return ph.cpu().numpy()


def _phasor_rel_l2(theta_gpu, p_ref):
    return np.linalg.norm(np.exp(1j * theta_gpu.astype(np.float64)) - p_ref) / np.linalg.norm(p_ref)


@pytest.mark.parametrize("method", [0, 1])
@pytest.mark.parametrize("n", [128, 512])
def test_gs_kinoform_and_restart_parity(api, oracle, method, n):
    cfg = W.CONFIGS["c5"].scaled(n)
    z = cfg.zs[0] * n / 8192                           # N pitch^2/(lambda z) = 0.718 as in c5
    amp_src, amp_dst, phi0 = W.gs_inputs_c5(cfg)
    # iters = 0: the kinoform (section 7.1)
    th = _gs_gpu(api, method, amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, 0)
    p = oracle.gs_init(method, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert _phasor_rel_l2(th, p) <= REL_L2
    assert th.min() >= -np.pi - 1e-6 and th.max() <= np.pi + 1e-6
    # restart parity along the oracle's trajectory: from the image-plane phase of
    # iteration t, one init + one loop pass on both sides
    for t in range(20):
        p, G = oracle.gs_iter(method, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z, want_G=True)
        if t in (0, 1, 5, 10, 19):
            phi_t = np.angle(G).astype(np.float32)
            th = _gs_gpu(api, method, amp_src, amp_dst, phi_t, cfg.pitch, cfg.lam, z, 1)
            pr = oracle.gs_init(method, amp_dst, phi_t, cfg.pitch, cfg.pitch, cfg.lam, z)
            pr = oracle.gs_iter(method, amp_src, amp_dst, pr, cfg.pitch, cfg.pitch, cfg.lam, z)
            assert _phasor_rel_l2(th, pr) <= REL_L2, "restart at t=%d" % t


@pytest.mark.parametrize("method", [0, 1])
@pytest.mark.parametrize("shape", [(2048, 2048), (4096, 4096), (4096, 64), (64, 4096), (8192, 64), (64, 8192)])
def test_gs_restart_parity_long_transforms(api, oracle, method, shape):
    """The GS load / store modes (amp * exp(i phi) load, phasor x amplitude store, atan2 store) on the tile shapes of
    the 4096- .. 16384-point transforms, full field: kinoform (iters = 0) and one-iteration restart from the
    oracle's state after its first loop pass."""
    cfg = W.CONFIGS["c5"]
    ny, nx = shape
    z = cfg.zs[0] * max(shape) / 8192
    amp_src, amp_dst, phi0 = W.gs_inputs(shape, 7)
    th = _gs_gpu(api, method, amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, 0)
    p = oracle.gs_init(method, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert _phasor_rel_l2(th, p) <= REL_L2, "kinoform %s" % (shape,)
    # a phasor is ill-conditioned where the field is nearly zero (error e at amplitude a moves it by e/a): the
    # maximum is only bounded loosely
    assert np.max(np.abs(np.exp(1j * th.astype(np.float64)) - p)) <= 5e-2
    p, G = oracle.gs_iter(method, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z, want_G=True)
    phi_t = np.angle(G).astype(np.float32)
    th = _gs_gpu(api, method, amp_src, amp_dst, phi_t, cfg.pitch, cfg.lam, z, 1)
    pr = oracle.gs_init(method, amp_dst, phi_t, cfg.pitch, cfg.pitch, cfg.lam, z)
    pr = oracle.gs_iter(method, amp_src, amp_dst, pr, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert _phasor_rel_l2(th, pr) <= REL_L2, "restart %s" % (shape,)


def test_gs_20_iteration_drift_reported(api, oracle, capsys):
    """the end-to-end phasor difference after 20 iterations is REPORTED, not gated at the
    single-propagation bar (fp32 and fp64 trajectories separate at near-zero amplitudes); only a loose sanity bound."""
    lines = []
    for method, n in ((0, 512), (1, 512)):
        cfg = W.CONFIGS["c5"].scaled(n)
        z = cfg.zs[0] * n / 8192
        amp_src, amp_dst, phi0 = W.gs_inputs_c5(cfg)
        th = _gs_gpu(api, method, amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, 20)
        ref = oracle.gs(method, amp_src, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z, 20)
        d = np.exp(1j * th.astype(np.float64)) - np.exp(1j * ref)
        rel, mx = np.linalg.norm(d) / np.sqrt(d.size), np.abs(d).max()
        lines.append("GS drift after 20 iterations, %s %d^2: phasor rel-L2 %.3e, max %.3e"
                     % ("Fresnel" if method == 0 else "ASM", n, rel, mx))
        assert rel < 5e-2
        if method == 0:
            # what an ordinary single-precision pipeline does on the SAME inputs: numpy's complex64 FFT, spectra built in
            # fp64 (test-side restatement of Listing 8, not product code).  The loop amplifies rounding differences at
            # near-zero amplitudes, so the drift depends on the inputs; this line is the yardstick for the one above.
            c64 = _gs_fresnel_numpy_c64(amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, 20)
            d = c64 - np.exp(1j * ref)
            rel64, mx64 = np.linalg.norm(d) / np.sqrt(d.size), np.abs(d).max()
            lines.append("   same inputs, plain complex64 numpy pipeline (fp64-built spectra):  phasor rel-L2 %.3e, max %.3e"
                         % (rel64, mx64))
            assert rel <= 2.0 * rel64          # the CUDA path does not drift more than an ordinary fp32 pipeline
    with capsys.disabled():
        print("\n" + "\n".join(lines))


def _gs_fresnel_numpy_c64(amp_src, amp_dst, phi0, pitch, lam, z, iters):
    n = amp_src.shape[0]

    def spectrum(zz):
        m = 2 * n
        d = np.arange(m); d = np.where(d < n, d, d - m).astype(np.float64)
        c1 = np.fft.fft(np.exp(1j * np.pi * (d * pitch) ** 2 / (lam * zz)))
        kz = zz / lam
        c = np.exp(2j * np.pi * (kz - np.floor(kz))) / (1j * lam * zz) * pitch * pitch
        return (np.outer(c1, c1) * c).astype(np.complex64)

    def prop(u, hh):
        big = np.zeros((2 * n, 2 * n), np.complex64); big[:n, :n] = u
        return np.fft.ifft2(np.fft.fft2(big) * hh)[:n, :n].astype(np.complex64)

    def phasor(u):
        a = np.abs(u); out = np.ones_like(u); nz = a > 0; out[nz] = u[nz] / a[nz]
        return out
    hm, hp = spectrum(-z), spectrum(+z)
    p = phasor(prop((amp_dst * np.exp(1j * phi0.astype(np.float64))).astype(np.complex64), hm))
    for _ in range(iters):
        q = phasor(prop((amp_src * p).astype(np.complex64), hp))
        p = phasor(prop((amp_dst * q).astype(np.complex64), hm))
    return p.astype(np.complex128)


def test_gs_error_curve_matches_oracle(api, oracle):
    # eps_t from the GPU trajectory equals the oracle's to <= 1e-5 at every t
    n = 256
    cfg = W.CONFIGS["c5"].scaled(n)
    z = cfg.zs[0] * n / 8192
    amp_src, amp_dst, phi0 = W.gs_inputs_c5(cfg)
    p = oracle.gs_init(0, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z)
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    errs = []
    for t in range(8):
        e_ref = oracle.gs_error(0, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z)
        th = _gs_gpu(api, 0, amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, t)
        field = _dev((amp_src * np.exp(1j * th.astype(np.float64))).astype(np.complex64))
        rec = torch.empty_like(field)
        api.cwo_fresnel_conv(plan, field, rec, z)
        e_gpu = float(torch.linalg.vector_norm(rec.abs() - _dev(amp_dst)) / torch.linalg.vector_norm(_dev(amp_dst)))
        assert abs(e_gpu - e_ref) <= 1e-5, (t, e_gpu, e_ref)
        errs.append(e_gpu)
        p = oracle.gs_iter(0, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert errs[-1] < errs[0]


def test_gs_c5_full_size(api, oracle):
    # 8192^2, 20 iterations in the bench configuration: runs, stays finite and in range, improves the
    # reconstruction; the kinoform step is spot-checked against the direct sum.
    cfg = W.CONFIGS["c5"]
    n, z = cfg.N, cfg.zs[0]
    amp_src, amp_dst, phi0 = W.gs_inputs_c5(cfg)
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    d_src, d_dst = _dev(amp_src), _dev(amp_dst)

    def recon_error(theta):
        field = torch.polar(d_src, theta)
        rec = torch.empty_like(field)
        api.cwo_fresnel_conv(plan, field, rec, z)
        return float(torch.linalg.vector_norm(rec.abs() - d_dst) / torch.linalg.vector_norm(d_dst))

    th0 = _dev(phi0.copy())
    api.cwo_gs(plan, d_src, d_dst, z, 0, th0)
    torch.cuda.synchronize()
    r = np.random.default_rng(3)
    ms = r.integers(0, n, 32); ns = r.integers(0, n, 32)
    G0 = (amp_dst.astype(np.float64) * np.exp(1j * phi0.astype(np.float64)))
    ref = oracle.fresnel_points(G0, cfg.pitch, cfg.pitch, cfg.lam, -z, ms, ns)
    got = np.exp(1j * th0.cpu().numpy()[ns, ms].astype(np.float64))
    pref = ref / np.abs(ref)
    # phasors: an error e of the field at amplitude a moves the phasor by e/a, so weigh by the sample's amplitude
    wgt = np.minimum(1.0, np.abs(ref) / np.abs(ref).max() * 4)
    assert np.linalg.norm((got - pref) * wgt) / np.linalg.norm(pref * wgt) <= REL_L2
    assert np.max(np.abs(got - pref) * wgt) <= MAX_ABS
    e0 = recon_error(th0)
    th = _dev(phi0.copy())
    api.cwo_gs(plan, d_src, d_dst, z, cfg.iters, th)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(th).all()) and float(th.abs().max()) <= np.pi + 1e-6
    assert recon_error(th) < e0


# ---------------------------------------------------------------- boundary -------------------------------------

def test_error_codes(api):
    plan = api.cwo_plan(64, 64, 1e-5, 633e-9)
    u = torch.zeros((64, 64), dtype=torch.complex64, device="cuda")
    with pytest.raises(api.CwoError) as e:
        api.cwo_fresnel_conv(plan, u, u, 0.0)
    assert e.value.code == api.CWO_EINVAL
    L = api.lib()
    assert L.cwo_asm(plan._h, u.data_ptr(), u.data_ptr(), 0.1) in (api.CWO_OK, api.CWO_EWORKSPACE)
    plan2 = api.cwo_plan(64, 64, 1e-5, 633e-9)
    assert L.cwo_asm(plan2._h, u.data_ptr(), u.data_ptr(), 0.1) == api.CWO_EWORKSPACE
    assert L.cwo_asm(plan2._h, u.data_ptr() + 8, u.data_ptr(), 0.1) == api.CWO_EINVAL
    assert L.cwo_asm(plan2._h, u.data_ptr(), u.data_ptr(), float("nan")) == api.CWO_EINVAL
    with pytest.raises(api.CwoError):
        api.cwo_plan(48, 64, 1e-5, 633e-9)
    big = api.cwo_plan(16384, 32, 1e-5, 633e-9)
    ub = torch.zeros((32, 16384), dtype=torch.complex64, device="cuda")
    with pytest.raises(api.CwoError):
        api.cwo_fresnel_conv(big, ub, ub, 0.1)      # 2*16384 exceeds the supported transform length
    assert plan.launch_count >= 2


def test_overlapping_buffers_are_refused(api):
    """include/cwo.h, Aliasing: exact in-place is allowed; partial overlap of an output with an input, or of a field with
    the workspace, returns CWO_EINVAL before anything is enqueued (launch count unchanged)."""
    n = 64
    fb = 8 * n * n
    L = api.lib()
    plan = api.cwo_plan(n, n, 1e-5, 633e-9)
    pool = torch.zeros(8 * n * n, dtype=torch.complex64, device="cuda")       # room for fields and a workspace side by side
    base = pool.data_ptr()
    plan.set_workspace(pool.view(torch.uint8)[4 * fb:])                        # workspace = second half of the pool
    plan.bind_stream()
    u1, u2 = base, base + fb
    assert L.cwo_asm(plan._h, u1, u2, 0.1) == api.CWO_OK                       # disjoint neighbours
    assert L.cwo_asm(plan._h, u1, u1, 0.1) == api.CWO_OK                       # exactly in place
    count = plan.launch_count
    for call in (L.cwo_asm, L.cwo_fresnel_conv):
        assert call(plan._h, u1, u1 + 16, 0.1) == api.CWO_EINVAL               # shifted by two samples
        assert call(plan._h, u1 + fb // 2, u1, 0.1) == api.CWO_EINVAL          # half a field apart
        assert call(plan._h, u1, base + 4 * fb, 0.1) == api.CWO_EINVAL         # u2 is the start of the workspace
        assert call(plan._h, base + 4 * fb - 16, u1, 0.1) == api.CWO_EINVAL    # u1 runs into the workspace
    zs = (api.ctypes.c_double * 2)(0.1, 0.2)
    assert L.cwo_propagate_stack(plan._h, u1, zs, 2, u1) == api.CWO_EINVAL     # the stack is never in place
    assert L.cwo_propagate_stack(plan._h, u1 + fb, zs, 2, u1) == api.CWO_EINVAL   # plane 1 of out = u1
    assert L.cwo_propagate_stack(plan._h, u1, zs, 2, base + 3 * fb) == api.CWO_EINVAL   # plane 1 of out = workspace
    plan.set_option(api.CWO_OPT_GS_METHOD, api.CWO_GS_ASM)
    rb = 4 * n * n
    a, b, ph = base, base + rb, base + 2 * rb
    assert L.cwo_gs(plan._h, a, a, 0.1, 0, ph) == api.CWO_OK                   # the two amplitudes may coincide
    assert L.cwo_gs(plan._h, a, b, 0.1, 1, b) == api.CWO_EINVAL                # phase_out = amp_dst
    assert L.cwo_gs(plan._h, a, b, 0.1, 1, a + 16) == api.CWO_EINVAL
    assert L.cwo_scale255(plan._h, a, a, n * n) == api.CWO_OK
    count = plan.launch_count
    assert L.cwo_scale255(plan._h, a, a + 16, n * n) == api.CWO_EINVAL
    assert L.cwo_pls_cgh(plan._h, a, 4, a) == api.CWO_EINVAL                   # the hologram over its own point list
    assert plan.launch_count == count
    torch.cuda.synchronize()


def test_host_pipeline_matches_oracle(api, oracle):
    """api.HostPipeline (pinned host buffers, copies overlapped over three streams): every step's result is
    that step's propagation -- more steps than device buffers, so slots are reused."""
    cfg = W.CONFIGS["c3"].scaled(256)
    plan = api.cwo_plan(cfg.N, cfg.N, cfg.pitch, cfg.lam)
    hp = api.HostPipeline(plan, "asm", depth=2)
    fields = [_rand((cfg.N, cfg.N), 100 + i) for i in range(5)]
    zs = [0.01, -0.02, 0.1, 0.5, 0.03]
    pins = [torch.from_numpy(f).pin_memory() for f in fields]
    outs = [torch.empty((cfg.N, cfg.N), dtype=torch.complex64).pin_memory() for _ in fields]
    cur = torch.cuda.current_stream()
    hp.start_after(cur)
    for p, o, z in zip(pins, outs, zs):
        hp.submit(p, o, z)
    hp.join(cur)
    torch.cuda.synchronize()
    for f, o, z in zip(fields, outs, zs):
        _assert_parity(o.numpy(), oracle.asm(f, cfg.pitch, cfg.pitch, cfg.lam, z), "host pipeline z=%g" % z)


# ---------------------------------------------------------------- launch-structure variants --------------------

@pytest.mark.parametrize("n", [1024, 2048, 4096])
def test_asm_and_fresnel_without_pipeline_option(api, oracle, n):
    """CWO_OPT_PIPELINE = 0 (one CTA per tile everywhere) computes the same propagations as the default."""
    cfg = W.CONFIGS["c3"].scaled(n)
    u1 = W.make_field(cfg)
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    plan.set_option(api.CWO_OPT_PIPELINE, 0)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, 0.03)
    torch.cuda.synchronize()
    _assert_parity(d2.cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, 0.03), "asm %d no pipeline" % n)
    if n <= 2048:
        m = n // 2
        v1 = np.ascontiguousarray(u1[:m, :m])
        planf = api.cwo_plan(m, m, 8e-6, 532e-9)
        planf.set_option(api.CWO_OPT_PIPELINE, 0)
        e1 = _dev(v1); e2 = torch.empty_like(e1)
        z = 0.2 * m / 1024
        api.cwo_fresnel_conv(planf, e1, e2, z)
        torch.cuda.synchronize()
        _assert_parity(e2.cpu().numpy(), oracle.fresnel_conv(v1, 8e-6, 8e-6, 532e-9, z), "fresnel %d no pipeline" % m)


def test_stack_batching_edges(api, oracle):
    """Batched stack launches: a batch remainder (5 planes, room for 3 per batch), the minimum workspace (one
    plane in flight: unbatched launches) and the pipeline option off all give the planes of independent cwo_asm."""
    n = 1024
    cfg = W.CONFIGS["c4"].scaled(n)
    u1 = W.make_field(cfg)
    zs = [0.001, 0.004, -0.002, 0.03, 0.064]
    ref = [oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, z) for z in zs]
    f = 8 * n * n
    for ws_planes, pipeline in ((4, 1), (2, 1), (17, 1), (4, 0)):
        plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
        plan.set_option(api.CWO_OPT_PIPELINE, pipeline)
        tables = plan.workspace_bytes(api.CWO_OP_STACK, len(zs)) - (1 + len(zs)) * f      # the planes' phase tables
        plan.set_workspace(torch.empty(ws_planes * f + tables, dtype=torch.uint8, device="cuda"))
        out = torch.empty((len(zs), n, n), dtype=torch.complex64, device="cuda")
        arr = (api.ctypes.c_double * len(zs))(*zs)
        plan.bind_stream()
        rc = api.lib().cwo_propagate_stack(plan._h, _dev(u1).data_ptr(), arr, len(zs), out.data_ptr())
        assert rc == 0
        torch.cuda.synchronize()
        for k in range(len(zs)):
            _assert_parity(out[k].cpu().numpy(), ref[k], "stack ws=%d planes pipeline=%d plane %d" % (ws_planes, pipeline, k))
    # below the minimum: refused, nothing enqueued
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    plan.set_workspace(torch.empty(f, dtype=torch.uint8, device="cuda"))
    out = torch.empty((1, n, n), dtype=torch.complex64, device="cuda")
    arr = (api.ctypes.c_double * 1)(0.01)
    assert api.lib().cwo_propagate_stack(plan._h, _dev(u1).data_ptr(), arr, 1, out.data_ptr()) == api.CWO_EWORKSPACE


@pytest.mark.parametrize("n", [256, 1024])
def test_stack_calls_back_to_back_on_one_workspace(api, oracle, n):
    """Two stack calls with different plane counts enqueued back to back on ONE workspace sized for the first: the
    second call's phase tables land where the first call's planes in flight were (the tables sit behind the planes),
    so its table kernel must not start writing before the first call's last kernel has finished reading (it is an
    ordinary, fully ordered launch when the tables live in the workspace).  Also a larger workspace than 64 planes' worth:
    the batch is clamped to 64."""
    cfg = W.CONFIGS["c4"].scaled(n)
    u1 = W.make_field(cfg)
    za, zb = [0.001, 0.004, -0.002], [0.002 * (k + 1) for k in range(7)]
    f = 8 * n * n
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    plan.set_workspace(torch.empty(plan.workspace_bytes(api.CWO_OP_STACK, len(za)) + 4096 * len(zb), dtype=torch.uint8, device="cuda"))
    d1 = _dev(u1)
    oa = torch.empty((len(za), n, n), dtype=torch.complex64, device="cuda")
    ob = torch.empty((len(zb), n, n), dtype=torch.complex64, device="cuda")
    plan.bind_stream()
    for rep in range(3):
        oa.zero_(); ob.zero_()
        assert api.lib().cwo_propagate_stack(plan._h, d1.data_ptr(), (api.ctypes.c_double * len(za))(*za), len(za), oa.data_ptr()) == 0
        assert api.lib().cwo_propagate_stack(plan._h, d1.data_ptr(), (api.ctypes.c_double * len(zb))(*zb), len(zb), ob.data_ptr()) == 0
        torch.cuda.synchronize()
        for k in (0, len(za) - 1):
            _assert_parity(oa[k].cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, za[k]), "first call, plane %d" % k)
        for k in (0, len(zb) - 1):
            _assert_parity(ob[k].cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, zb[k]), "second call, plane %d" % k)
    if n == 1024:     # a workspace for 80 planes in flight: batches of at most 64 (70 planes = 64 + 6)
        zs = [0.0005 * (k + 1) for k in range(70)]
        plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
        plan.set_workspace(torch.empty(81 * f + 4 * 70 * (2 * n + 1) + 256, dtype=torch.uint8, device="cuda"))
        out = torch.empty((len(zs), n, n), dtype=torch.complex64, device="cuda")
        plan.bind_stream()
        assert api.lib().cwo_propagate_stack(plan._h, d1.data_ptr(), (api.ctypes.c_double * len(zs))(*zs), len(zs), out.data_ptr()) == 0
        torch.cuda.synchronize()
        for k in (0, 63, 64, 69):
            _assert_parity(out[k].cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, zs[k]), "plane %d of 70" % k)


def test_back_to_back_calls_on_a_side_stream(api, oracle):
    """Programmatic dependent launch keeps stream order: alternating ASM / Fresnel calls with changing z, enqueued
    back to back on a non-default stream without synchronising, each read its predecessor's output."""
    n = 1024
    cfg = W.CONFIGS["c3"].scaled(n)
    u1 = W.make_field(cfg)
    s = torch.cuda.Stream()
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    a = _dev(u1); b = torch.empty_like(a); c = torch.empty_like(a)
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        api.cwo_asm(plan, a, b, 0.01)
        api.cwo_asm(plan, b, c, 0.02)          # semigroup: c = P(0.03) a
        api.cwo_asm(plan, c, b, -0.03)         # b = a
        api.cwo_fresnel_conv(plan, b, c, 0.4)
    s.synchronize()
    _assert_parity(b.cpu().numpy(), u1.astype(np.complex128), "chain back to the input")
    _assert_parity(c.cpu().numpy(), oracle.fresnel_conv(u1, cfg.pitch, cfg.pitch, cfg.lam, 0.4), "fresnel after the chain")


# ---------------------------------------------------------------- randomised sweep -------------------------------


def test_workspace_is_recorded_on_every_stream_it_is_used_on(api, oracle):
    """The binding's workspace is a torch tensor: when it is regrown, the old block goes back to the caching allocator,
    which may only reuse it once the kernels enqueued on EVERY stream the plan ran on are done.  The plan records the
    workspace on each stream it is bound to (Plan.bind_stream), not on whatever stream is current when it regrows."""
    u1 = _rand((512, 512), 71)
    px, lam, z = 4e-6, 633e-9, 0.01
    plan = api.cwo_plan(512, 512, px, lam)
    d1 = _dev(u1); d2 = torch.empty_like(d1); d3 = torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, z)                          # workspace allocated and used under the default stream
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    ws0 = plan._ws
    with torch.cuda.stream(side):
        api.cwo_asm(plan, d1, d2, -z)                     # the same block, now used on the side stream
        assert side.cuda_stream in plan._ws_streams
    api.cwo_fresnel_conv(plan, d1, d3, z)                 # regrows under the default stream while `side` may still run
    assert plan._ws is not ws0 and torch.cuda.current_stream().cuda_stream in plan._ws_streams
    assert side.cuda_stream not in plan._ws_streams       # the new block has not been used there
    torch.cuda.synchronize()
    _assert_parity(d2.cpu().numpy(), oracle.asm(u1, px, px, lam, -z), "asm on the side stream")
    _assert_parity(d3.cpu().numpy(), oracle.fresnel_conv(u1, px, px, lam, z), "fresnel after the regrowth")


@pytest.mark.parametrize("seed", range(16))
def test_random_shapes_and_parameters(api, oracle, seed):
    """Seeded sweep over shapes (powers of two, Nx != Ny allowed), pitches, wavelengths and distances of both
    signs, for both propagations, including in-place calls."""
    r = np.random.default_rng(20240 + seed)
    lx, ly = int(r.integers(5, 12)), int(r.integers(5, 12))
    if lx + ly > 21:                      # keep the fp64 oracle to seconds
        ly = 21 - lx
    nx, ny = 1 << lx, 1 << ly
    lam = float(r.choice([405e-9, 532e-9, 633e-9, 1064e-9]))
    px, py = float(r.uniform(2.0, 12.0)) * lam * 2, float(r.uniform(2.0, 12.0)) * lam * 2
    z = float(r.choice([-1, 1])) * float(r.uniform(0.002, 0.3))
    u1 = _rand((ny, nx), 900 + seed)
    inplace = bool(seed & 1)
    _assert_parity(_gpu_asm(api, u1, px, py, lam, z, inplace=inplace), oracle.asm(u1, px, py, lam, z),
                   "asm %dx%d px=%g py=%g lam=%g z=%g" % (ny, nx, px, py, lam, z))
    if lx <= 10 and ly <= 10:
        _assert_parity(_gpu_fresnel(api, u1, px, py, lam, z, inplace=inplace), oracle.fresnel_conv(u1, px, py, lam, z),
                       "fresnel %dx%d px=%g py=%g lam=%g z=%g" % (ny, nx, px, py, lam, z))


def test_asm_16384_square_plane_wave_and_roundtrip(api):
    """Largest supported ASM (16384 x 16384, the cluster row kernel without padding), checked without the oracle:
    a plane wave is an eigenfunction, u2 = H(k0, l0) u1 with H from Eq.(16) in double; z then -z returns the input."""
    n, px, lam, z = 16384, 4e-6, 633e-9, 0.05
    k0, l0 = 37, -1234
    j = torch.arange(n, device="cuda", dtype=torch.float64)
    phx = torch.remainder(k0 * j, n) * (2 * np.pi / n)
    phy = torch.remainder(l0 * j, n) * (2 * np.pi / n)
    u1 = torch.polar(torch.ones((n, n), device="cuda", dtype=torch.float32),
                     (phy[:, None] + phx[None, :]).to(torch.float32)).contiguous()
    del phx, phy
    plan = api.cwo_plan(n, n, px, lam)
    u2 = torch.empty_like(u1)
    api.cwo_asm(plan, u1, u2, z)
    torch.cuda.synchronize()
    fx, fy = k0 / (n * px), l0 / (n * px)
    w = 1.0 / lam ** 2 - (fx * fx + fy * fy)
    ph = z * np.sqrt(w)
    H = np.exp(2j * np.pi * (ph - np.floor(ph)))
    err = torch.linalg.vector_norm(u2 - complex(H) * u1) / torch.linalg.vector_norm(u1)
    assert float(err) <= REL_L2, "plane wave eigenfunction rel-L2 %.3e" % float(err)
    api.cwo_asm(plan, u2, u2, -z)                       # in place, back
    torch.cuda.synchronize()
    err = torch.linalg.vector_norm(u2 - u1) / torch.linalg.vector_norm(u1)
    assert float(err) <= REL_L2, "round trip rel-L2 %.3e" % float(err)


# ---------------------------------------------------------------- zero-expanded ASM --------------

def _gpu_asm_pad2x(api, u1, px, py, lam, z, inplace=False):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, px, lam)
    if px != py:
        plan.set_pitch_xy(px, py)
    plan.set_option(api.CWO_OPT_ASM_PAD2X, 1)
    d1 = _dev(u1)
    d2 = d1 if inplace else torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


@pytest.mark.parametrize("shape", [(32, 32), (64, 256), (512, 128), (1024, 1024), (2048, 512), (256, 4096), (2048, 2048)])
def test_asm_pad2x_sizes(api, oracle, shape):
    u1 = _rand(shape, 31)
    px, py, lam = 4e-6, 5e-6, 633e-9
    for z, inplace in ((0.01, False), (-0.004, True)):
        _assert_parity(_gpu_asm_pad2x(api, u1, px, py, lam, z, inplace), oracle.asm_pad2x(u1, px, py, lam, z),
                       "asm pad2x %s z=%g" % (shape, z))


def test_asm_pad2x_c1_evanescent_and_option_scope(api, oracle):
    cfg = W.CONFIGS["c1"]
    u1 = W.make_field(cfg)
    _assert_parity(_gpu_asm_pad2x(api, u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]),
                   oracle.asm_pad2x(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]), "c1 pad2x")
    # pitch < lambda / sqrt(2): evanescent bins on the expanded grid (fp64 per-sample path)
    v1 = _rand((64, 64), 33)
    _assert_parity(_gpu_asm_pad2x(api, v1, 0.3e-6, 0.3e-6, 633e-9, 5e-6), oracle.asm_pad2x(v1, 0.3e-6, 0.3e-6, 633e-9, 5e-6),
                   "pad2x evanescent")
    # the option changes cwo_asm only: the stack still gives the circular form; sizes above 8192 are refused
    plan = api.cwo_plan(256, 256, cfg.pitch, cfg.lam)
    plan.set_option(api.CWO_OPT_ASM_PAD2X, 1)
    out = torch.empty((1, 256, 256), dtype=torch.complex64, device="cuda")
    api.cwo_propagate_stack(plan, _dev(u1), [cfg.zs[0]], out)
    torch.cuda.synchronize()
    _assert_parity(out[0].cpu().numpy(), oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, cfg.zs[0]), "stack stays circular")
    big = api.cwo_plan(16384, 32, cfg.pitch, cfg.lam)
    with pytest.raises(api.CwoError):
        big.set_option(api.CWO_OPT_ASM_PAD2X, 1)


def test_asm_pad2x_toggled_on_one_plan(api, oracle):
    """circular -> zero-expanded -> circular on ONE plan (the per-z tables double in size with the option)."""
    u1 = _rand((512, 1024), 35)
    px, lam, z = 4e-6, 633e-9, 0.02
    plan = api.cwo_plan(1024, 512, px, lam)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    for pad in (0, 1, 0, 1):
        plan.set_option(api.CWO_OPT_ASM_PAD2X, pad)
        for zz in (z, -0.5 * z):
            api.cwo_asm(plan, d1, d2, zz)
            torch.cuda.synchronize()
            ref = (oracle.asm_pad2x if pad else oracle.asm)(u1, px, px, lam, zz)
            _assert_parity(d2.cpu().numpy(), ref, "pad=%d z=%g" % (pad, zz))


def test_asm_pad2x_4096(api, oracle):
    cfg = W.CONFIGS["c3"]
    u1 = W.make_field(cfg)
    _assert_parity(_gpu_asm_pad2x(api, u1, cfg.pitch, cfg.pitch, cfg.lam, 0.1), oracle.asm_pad2x(u1, cfg.pitch, cfg.pitch, cfg.lam, 0.1),
                   "asm pad2x 4096")


# ---------------------------------------------------------------- shifted / band-limited ASM ---------

def _gpu_asm_shifted(api, u1, px, py, lam, z, ox=0.0, oy=0.0):
    ny, nx = u1.shape
    plan = api.cwo_plan(nx, ny, px, lam)
    if px != py:
        plan.set_pitch_xy(px, py)
    plan.set_option(api.CWO_OPT_ASM_BAND_LIMIT, 1)
    plan.set_offset(ox, oy)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, z)
    torch.cuda.synchronize()
    return d2.cpu().numpy()


@pytest.mark.parametrize("shape", [(64, 64), (128, 32), (256, 512), (1024, 1024), (512, 4096), (2048, 2048), (32, 16384)])
def test_asm_band_limited_and_shifted(api, oracle, shape):
    """Eq.(18)-(19): the band limit cuts part of the grid (z chosen so that the edge is at ~1/3 of the Nyquist
    frequency of the longer axis), on axis and with an offset of a non-integer number of pitches, both signs of z.
    Scalar tiles (< 256 points), lane-pair tiles and the single-lane 16384-point tile."""
    ny, nx = shape
    px, py, lam = 4e-6, 5e-6, 633e-9
    n = max(nx, ny)
    p = px if nx >= ny else py
    z = n * p * p / lam * 1.5                            # band edge = Nyquist / 3 along the longer axis
    u1 = _rand(shape, 51)
    for zz, ox, oy in ((z, 0.0, 0.0), (-z, 0.0, 0.0), (z, 37.3 * px, -11.6 * py)):
        ref = oracle.asm_shifted(u1, px, py, lam, zz, ox, oy)
        assert np.linalg.norm(ref) < 0.9 * np.linalg.norm(u1)            # the band really removes something
        _assert_parity(_gpu_asm_shifted(api, u1, px, py, lam, zz, ox, oy), ref, "shifted asm %s z=%g O=(%g,%g)" % (shape, zz, ox, oy))


def test_asm_band_limited_fp64_path_and_option_off(api, oracle):
    # pitch < lambda / sqrt(2): the per-sample fp64 transfer function (evanescent bins) with the band limit and the ramp
    u1 = _rand((64, 64), 53)
    d, lam, z = 0.3e-6, 633e-9, 2e-5
    _assert_parity(_gpu_asm_shifted(api, u1, d, d, lam, z, 3.2 * d, -1.5 * d), oracle.asm_shifted(u1, d, d, lam, z, 3.2 * d, -1.5 * d),
                   "shifted asm, fp64 path")
    # the offset has no effect while the option is off
    plan = api.cwo_plan(64, 64, 4e-6, lam)
    plan.set_offset(1e-4, 1e-4)
    d1 = _dev(u1); d2 = torch.empty_like(d1)
    api.cwo_asm(plan, d1, d2, 0.01)
    torch.cuda.synchronize()
    _assert_parity(d2.cpu().numpy(), oracle.asm(u1, 4e-6, 4e-6, lam, 0.01), "option off")


@pytest.mark.parametrize("n,pipeline", [(256, 1), (1024, 1), (1024, 0)])
def test_band_limit_and_offset_are_cwo_asm_only(api, oracle, n, pipeline):
    """include/cwo.h: CWO_OPT_ASM_BAND_LIMIT and cwo_plan_set_offset change cwo_asm only.  With both set, the stack
    (one launch pair per batch at 1024, plane by plane otherwise) and GS with the ASM propagator must give exactly what
    they give without them -- at distances where the band of Eq.(18) would cut most of the grid and differs per plane."""
    px, lam = 4e-6, 633e-9
    zb = n * px * px / lam                                 # band edge = Nyquist / 2 at 1.0 zb, Nyquist / 6 at 3 zb
    zs = [0.7 * zb, 3.0 * zb, -1.5 * zb, 2.2 * zb, 0.4 * zb]
    u1 = _rand((n, n), 61)
    outs = []
    for band in (0, 1):
        plan = api.cwo_plan(n, n, px, lam)
        plan.set_option(api.CWO_OPT_PIPELINE, pipeline)
        if band:
            plan.set_option(api.CWO_OPT_ASM_BAND_LIMIT, 1)
            plan.set_offset(13.4 * px, -7.7 * px)
        out = torch.empty((len(zs), n, n), dtype=torch.complex64, device="cuda")
        api.cwo_propagate_stack(plan, _dev(u1), zs, out)
        torch.cuda.synchronize()
        outs.append(out.cpu().numpy())
    assert np.array_equal(outs[0], outs[1])
    for k in (0, 1, 4):
        _assert_parity(outs[1][k], oracle.asm(u1, px, px, lam, zs[k]), "stack plane %d with the band option set" % k)
    amp_src, amp_dst, phi0 = W.gs_inputs((n, n), 9)
    phases = []
    for band in (0, 1):
        plan = api.cwo_plan(n, n, px, lam)
        plan.set_option(api.CWO_OPT_PIPELINE, pipeline)
        plan.set_option(api.CWO_OPT_GS_METHOD, api.CWO_GS_ASM)
        if band:
            plan.set_option(api.CWO_OPT_ASM_BAND_LIMIT, 1)
            plan.set_offset(13.4 * px, -7.7 * px)
        ph = _dev(phi0.astype(np.float32))
        api.cwo_gs(plan, _dev(amp_src), _dev(amp_dst), 3.0 * zb, 2, ph)
        torch.cuda.synchronize()
        phases.append(ph.cpu().numpy())
    assert np.array_equal(phases[0], phases[1])


@pytest.mark.parametrize("shape", [(64, 64), (256, 512), (1024, 1024), (4096, 4096)])
def test_asm_pad2x_with_band_limit(api, oracle, shape):
    """Zero expansion and the band limit together (the band-limited method of Eq.(18) as its authors use it: on the 2N grid):
    the oracle's band-limited ASM on the field expanded with zeros, cropped.  4096: the prefetching padded column kernel."""
    ny, nx = shape
    px, lam = 4e-6, 633e-9
    z = 2 * max(nx, ny) * px * px / lam * 1.5              # band edge = Nyquist / 3 on the expanded grid
    u1 = _rand(shape, 63)
    big = np.zeros((2 * ny, 2 * nx), dtype=np.complex64); big[:ny, :nx] = u1
    cases = ((z, 0.0, 0.0), (-z, 21.3 * px, -9.6 * px)) if nx < 4096 else ((z, 21.3 * px, -9.6 * px),)
    for zz, ox, oy in cases:
        ref = oracle.asm_shifted(big, px, px, lam, zz, ox, oy)[:ny, :nx]
        plan = api.cwo_plan(nx, ny, px, lam)
        plan.set_option(api.CWO_OPT_ASM_PAD2X, 1)
        plan.set_option(api.CWO_OPT_ASM_BAND_LIMIT, 1)
        plan.set_offset(ox, oy)
        d1 = _dev(u1); d2 = torch.empty_like(d1)
        api.cwo_asm(plan, d1, d2, zz)
        torch.cuda.synchronize()
        _assert_parity(d2.cpu().numpy(), ref, "pad2x + band limit %s z=%g O=(%g,%g)" % (shape, zz, ox, oy))


@pytest.mark.parametrize("method", [0, 1])
def test_gs_with_zeros_in_the_target_amplitude(api, oracle, method):
    """A target image with a black region (amp_dst == 0 there), 1024^2 (the packed TMA row store of the phasor x amplitude
    mode): kinoform and one-iteration restart against the oracle; and an all-black target, where every propagated field
    is exactly zero and phasor(0) = 1 (cwo.h) must give phase 0 everywhere, not NaN."""
    n = 1024
    cfg = W.CONFIGS["c5"]
    z = cfg.zs[0] * n / 8192
    amp_src, amp_dst, phi0 = W.gs_inputs((n, n), 11)
    amp_dst = amp_dst.copy(); amp_dst[: n // 2, :] = 0.0; amp_dst[:, 100:164] = 0.0
    th = _gs_gpu(api, method, amp_src, amp_dst, phi0, cfg.pitch, cfg.lam, z, 0)
    p = oracle.gs_init(method, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert _phasor_rel_l2(th, p) <= REL_L2
    p, G = oracle.gs_iter(method, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, z, want_G=True)
    phi_t = np.angle(G).astype(np.float32)
    th = _gs_gpu(api, method, amp_src, amp_dst, phi_t, cfg.pitch, cfg.lam, z, 1)
    pr = oracle.gs_init(method, amp_dst, phi_t, cfg.pitch, cfg.pitch, cfg.lam, z)
    pr = oracle.gs_iter(method, amp_src, amp_dst, pr, cfg.pitch, cfg.pitch, cfg.lam, z)
    assert _phasor_rel_l2(th, pr) <= REL_L2
    black = np.zeros_like(amp_dst)
    for iters in (0, 2):
        th = _gs_gpu(api, method, amp_src, black, phi0, cfg.pitch, cfg.lam, z, iters)
        assert np.all(th == 0.0), "all-black target, iters=%d" % iters
        assert np.all(oracle.gs(method, amp_src, black, phi0, cfg.pitch, cfg.pitch, cfg.lam, z, iters) == 0.0)


# ---------------------------------------------------------------- intensity stack --------------------

@pytest.mark.parametrize("n,pipeline", [(256, 1), (1024, 1), (1024, 0), (2048, 1)])
def test_stack_intensity(api, oracle, n, pipeline):
    """CWO_OPT_STACK_INTENSITY: float |u|^2 planes (Eq.(20)) from the batched and the unbatched launches."""
    cfg = W.CONFIGS["c4"].scaled(n)
    u1 = W.make_field(cfg)
    zs = [0.001, 0.0047, -0.002, 0.064, 0.03]
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    plan.set_option(api.CWO_OPT_PIPELINE, pipeline)
    plan.set_option(api.CWO_OPT_STACK_INTENSITY, 1)
    out = torch.empty((len(zs), n, n), dtype=torch.float32, device="cuda")
    api.cwo_propagate_stack(plan, _dev(u1), zs, out)
    torch.cuda.synchronize()
    ref = oracle.stack_intensity(u1, cfg.pitch, cfg.pitch, cfg.lam, zs)
    got = out.cpu().numpy().astype(np.float64)
    for k in range(len(zs)):
        rel = np.linalg.norm(got[k] - ref[k]) / np.linalg.norm(ref[k])
        mx = np.max(np.abs(got[k] - ref[k])) / np.max(ref[k])
        # |u|^2 doubles the relative error of u: bars 2 x (2e-5, 1e-4)
        assert rel <= 2 * REL_L2 and mx <= 2 * MAX_ABS, "intensity plane %d: %.3e %.3e" % (k, rel, mx)


# ---------------------------------------------------------------- the calls only enqueue: CUDA graph capture ----------

def test_calls_capture_into_a_cuda_graph_and_replay(api, oracle):
    """include/cwo.h: every propagation call only enqueues kernels on the plan's stream (no allocation, no
    synchronisation, no copy), so a sequence of calls can be captured into a CUDA graph and replayed on new data."""
    n = 512
    cfg = W.CONFIGS["c3"].scaled(n)
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    for op in (api.CWO_OP_ASM, api.CWO_OP_FRESNEL, api.CWO_OP_GS, api.CWO_OP_STACK):
        plan.ensure_workspace(op, 3)
    amp_src, amp_dst, phi0 = W.gs_inputs((n, n), 3)
    a = torch.empty((n, n), dtype=torch.complex64, device="cuda")
    b = torch.empty_like(a); c = torch.empty_like(a)
    st = torch.empty((3, n, n), dtype=torch.complex64, device="cuda")
    d_src, d_dst, d_phi = _dev(amp_src), _dev(amp_dst), _dev(phi0)
    zs = [0.002, 0.004, -0.003]
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        # warm-up outside the capture (lazy module loading is not capturable)
        api.cwo_asm(plan, a, b, 0.01); api.cwo_fresnel_conv(plan, b, c, 0.4)
        api.cwo_propagate_stack(plan, a, zs, st); api.cwo_gs(plan, d_src, d_dst, 0.02, 1, d_phi)
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            api.cwo_asm(plan, a, b, 0.01)
            api.cwo_fresnel_conv(plan, b, c, 0.4)
            api.cwo_propagate_stack(plan, a, zs, st)
            api.cwo_gs(plan, d_src, d_dst, 0.02, 2, d_phi)
    for seed in (61, 62):
        u1 = _rand((n, n), seed)
        a.copy_(_dev(u1)); d_phi.copy_(_dev(phi0))
        g.replay()
        torch.cuda.synchronize()
        ref_b = oracle.asm(u1, cfg.pitch, cfg.pitch, cfg.lam, 0.01)
        _assert_parity(b.cpu().numpy(), ref_b, "graph: asm")
        _assert_parity(c.cpu().numpy(), oracle.fresnel_conv(b.cpu().numpy(), cfg.pitch, cfg.pitch, cfg.lam, 0.4), "graph: fresnel")
        ref_s = oracle.stack(u1, cfg.pitch, cfg.pitch, cfg.lam, zs)
        for k in range(3):
            _assert_parity(st[k].cpu().numpy(), ref_s[k], "graph: stack %d" % k)
        p = oracle.gs_init(0, amp_dst, phi0, cfg.pitch, cfg.pitch, cfg.lam, 0.02)
        for _ in range(2):
            p = oracle.gs_iter(0, amp_src, amp_dst, p, cfg.pitch, cfg.pitch, cfg.lam, 0.02)
        val = _phasor_rel_l2(d_phi.cpu().numpy(), p)
        print("MEASURED graph gs two iterations: phasor rel-L2 %.3e" % val)
        assert val <= REL_L2         # two iterations; measured 3.6e-6 on the B200 (SURVEY G5 allowed a drift of 5x)
