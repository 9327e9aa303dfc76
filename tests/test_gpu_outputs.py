"""Parity of Scale (Eq.(21)) and the point-light-source CGH (Eq.(23)) of the CUDA path against the fp64 oracle
(SURVEY 8(f) f4)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_parity import REL_L2, MAX_ABS, api   # noqa: E402,F401

LAM = 633e-9


def _points(n, seed, span, z0, dz):
    r = np.random.default_rng(seed)
    return np.stack([r.uniform(-span, span, n), r.uniform(-span, span, n), z0 + r.uniform(-dz, dz, n),
                     r.uniform(0.2, 1.0, n)], axis=1)


@pytest.mark.parametrize("shape,npts", [((64, 128), 1), ((256, 256), 333), ((16, 64), 70), ((512, 1024), 1200)])
def test_pls_cgh_matches_oracle(api, oracle, shape, npts):
    # sizes below and above the 128 x 32 tile, a ragged point count (chunks of 32), points off the grid,
    # phases up to ~1e4 cycles: element by element at the propagation bar
    ny, nx = shape
    px, py = 4e-6, 5e-6
    pts = _points(npts, 7 + npts, 1.5e-3, 0.2, 0.03)
    if npts == 70:
        pts[:, 2] *= -1                       # z_j < 0: same pattern (cos is even)
    plan = _plan_of_shape(api, nx, ny, px, py)
    out = torch.empty((ny, nx), dtype=torch.float32, device="cuda")
    api.cwo_pls_cgh(plan, torch.from_numpy(pts).cuda(), out)
    torch.cuda.synchronize()
    ref = oracle.pls_cgh(ny, nx, px, py, LAM, pts[:, 0], pts[:, 1], pts[:, 2], pts[:, 3])
    got = out.cpu().numpy().astype(np.float64)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert rel <= REL_L2 and np.abs(got - ref).max() <= MAX_ABS * np.abs(ref).max(), (rel, np.abs(got - ref).max())


def _plan_of_shape(api, nx, ny, px, py):
    # cwo_plan wants powers of two; the CGH call itself does not: take the enclosing power-of-two plan when the
    # shape is one, else skip (the C ABI ties the grid to the plan)
    def p2(v):
        return v & (v - 1) == 0
    if not (p2(nx) and p2(ny)):
        pytest.skip("plan grids are powers of two")
    plan = api.cwo_plan(nx, ny, px, LAM)
    if px != py:
        plan.set_pitch_xy(px, py)
    return plan


def test_pls_cgh_paper_sized_sampled(api, oracle):
    # the paper's List 3: 2048 x 2048 hologram, 11 646 points, pitch 4 um, 633 nm, 0.2 m; object within +-4 mm, offset
    # (1 cm, -2 mm).  The oracle evaluates 64 hologram rows (of 2048) in full
    n, npts = 2048, 11646
    pts = _points(npts, 3, 4e-3, 0.2, 4e-3)
    pts[:, 0] += 1e-2; pts[:, 1] -= 2e-3
    plan = api.cwo_plan(n, n, 4e-6, LAM)
    out = torch.empty((n, n), dtype=torch.float32, device="cuda")
    api.cwo_pls_cgh(plan, torch.from_numpy(pts).cuda(), out)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    rows = np.r_[0, 1, 31, 32, 33, n - 1, np.random.default_rng(4).integers(0, n, 58)]
    oracle.set_threads(oracle.max_threads())
    # the oracle on a 64 x 2048 strip: shift the points' y so that strip row r is hologram row rows[r]
    err2 = ref2 = 0.0; mx = pk = 0.0
    for r in rows:
        strip = oracle.pls_cgh(2, n, 4e-6, 4e-6, LAM, pts[:, 0], pts[:, 1] - (r - n // 2 + 1) * 4e-6, pts[:, 2], pts[:, 3])[0]
        d = got[r] - strip
        err2 += d @ d; ref2 += strip @ strip; mx = max(mx, np.abs(d).max()); pk = max(pk, np.abs(strip).max())
    oracle.set_threads(min(8, oracle.max_threads()))
    assert np.sqrt(err2 / ref2) <= REL_L2 and mx <= MAX_ABS * pk, (np.sqrt(err2 / ref2), mx, pk)


@pytest.mark.parametrize("n", [1, 5, 1000, 256 * 256 + 3, 2048 * 2048])
def test_scale255_matches_oracle(api, oracle, n):
    r = np.random.default_rng(n)
    a = (r.standard_normal(n) ** 2 * 37.0 - 3.0).astype(np.float32)
    plan = api.cwo_plan(256, 256, 4e-6, LAM)
    d = torch.from_numpy(a).cuda()
    o = torch.empty_like(d)
    api.cwo_scale255(plan, d, o)
    torch.cuda.synchronize()
    ref = oracle.scale255(a.astype(np.float64))
    got = o.cpu().numpy()
    assert np.abs(got - ref).max() <= 255 * 4e-7 * 8
    if n > 1:
        assert got.min() == 0.0 and got.max() == 255.0
        assert got[np.argmin(a)] == 0.0 and got[np.argmax(a)] == 255.0
    api.cwo_scale255(plan, d, d)              # in place, and a second call on the same plan (min/max cells reset)
    torch.cuda.synchronize()
    assert np.array_equal(d.cpu().numpy(), got)


def test_scale255_of_a_stack_intensity(api, oracle):
    # Listing 1/2 of the paper: Diffract -> Intensity -> Scale
    from paper_1107_5578_b200 import workloads as W
    cfg = W.CONFIGS["c4"].scaled(256)
    u1 = W.make_field(cfg)
    zs = list(cfg.zs[:3])
    plan = api.cwo_plan(256, 256, cfg.pitch, cfg.lam)
    plan.set_option(api.CWO_OPT_STACK_INTENSITY, 1)
    out = torch.empty((3, 256, 256), dtype=torch.float32, device="cuda")
    api.cwo_propagate_stack(plan, torch.from_numpy(u1).cuda(), zs, out)
    api.cwo_scale255(plan, out, out)
    torch.cuda.synchronize()
    ref = oracle.scale255(oracle.stack_intensity(u1, cfg.pitch, cfg.pitch, cfg.lam, zs))
    assert np.abs(out.cpu().numpy() - ref).max() <= 255 * 2e-5


def test_new_calls_capture_into_a_cuda_graph_and_replay(api, oracle):
    """cwo_fresnel_fourier, cwo_fresnel_shifted, cwo_pls_cgh and cwo_scale255 only enqueue (kernels and two memsets): a
    sequence of them is captured into a CUDA graph and replayed on new data."""
    from test_gpu_parity import _assert_parity, _dev, _rand
    n, p, lam = 512, 8e-6, 532e-9
    plan = api.cwo_plan(n, n, p, lam)
    plan.set_dst_pitch_xy(5e-6, 11e-6); plan.set_offset(2e-4, -1e-4)
    plan.ensure_workspace(api.CWO_OP_FRESNEL_SHIFTED)
    a = torch.empty((n, n), dtype=torch.complex64, device="cuda")
    b = torch.empty_like(a); c = torch.empty_like(a)
    holo = torch.empty((n, n), dtype=torch.float32, device="cuda"); holo8 = torch.empty_like(holo)
    pts = _points(50, 5, 1e-3, 0.2, 0.02)
    d_pts = torch.from_numpy(pts).cuda()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        api.cwo_fresnel_fourier(plan, a, b, 0.1); api.cwo_fresnel_shifted(plan, a, c, 0.1)
        api.cwo_pls_cgh(plan, d_pts, holo); api.cwo_scale255(plan, holo, holo8)
        s.synchronize()
        with torch.cuda.graph(g, stream=s):
            api.cwo_fresnel_fourier(plan, a, b, 0.1)
            api.cwo_fresnel_shifted(plan, a, c, -0.07)
            api.cwo_pls_cgh(plan, d_pts, holo)
            api.cwo_scale255(plan, holo, holo8)
    for seed in (71, 72):
        u1 = _rand((n, n), seed)
        a.copy_(_dev(u1))
        pts2 = _points(50, seed, 1e-3, 0.2, 0.02)
        d_pts.copy_(torch.from_numpy(pts2).cuda())
        g.replay()
        torch.cuda.synchronize()
        _assert_parity(b.cpu().numpy(), oracle.fresnel_fourier(u1, p, p, lam, 0.1), "graph: fourier")
        _assert_parity(c.cpu().numpy(), oracle.fresnel_shifted(u1, (p, p), (5e-6, 11e-6), lam, -0.07, o1=(2e-4, -1e-4)),
                       "graph: shifted")
        ref = oracle.pls_cgh(n, n, p, p, lam, pts2[:, 0], pts2[:, 1], pts2[:, 2], pts2[:, 3])
        got = holo.cpu().numpy().astype(np.float64)
        assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= REL_L2
        assert np.abs(holo8.cpu().numpy() - oracle.scale255(got)).max() <= 255 * 4e-6


# ---------------------------------------------------------------- intensity output of one propagation -----------------

def _rand_field(shape, seed):
    r = np.random.default_rng(seed)
    return (r.standard_normal(shape) + 1j * r.standard_normal(shape)).astype(np.complex64)


def _assert_intensity(got, ref, what):
    got = got.astype(np.float64)
    rel = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    mx = np.max(np.abs(got - ref)) / np.max(ref)
    # |u|^2 doubles the relative error of u: bars 2 x (2e-5, 1e-4), as for the intensity stack
    assert rel <= 2 * REL_L2 and mx <= 2 * MAX_ABS, "%s: rel-L2 %.3e max/peak %.3e" % (what, rel, mx)


@pytest.mark.parametrize("case", [
    ("asm", (64, 64)), ("asm", (256, 512)), ("asm", (1024, 1024)), ("asm", (64, 4096)), ("asm", (64, 8192)), ("asm", (32, 16384)),
    ("asm", (2048, 2048)), ("asm_pad2x", (256, 256)), ("asm_pad2x", (1024, 1024)), ("asm_pad2x", (64, 4096)),
    ("fresnel", (64, 64)), ("fresnel", (128, 32)), ("fresnel", (256, 512)), ("fresnel", (1024, 1024)), ("fresnel", (4096, 256)),
    ("fourier", (256, 512)), ("fourier", (1024, 1024)), ("shifted", (512, 256)), ("shifted", (1024, 1024))],
    ids=lambda c: "%s-%dx%d" % (c[0], c[1][0], c[1][1]))
def test_real_field_output_of_single_propagations(api, oracle, case):
    """CWO_OPT_OUT_REAL (the paper's Listing 1: Diffract -> Intensity; section 5: Amp, Re(), Im, Phase()): a float field of
    u2 from the last store of cwo_asm (circular and zero-expanded; scalar, lane-pair, pipelined and one-row tiles),
    cwo_fresnel_conv (three-pass form below 256, separable form above), cwo_fresnel_fourier and cwo_fresnel_shifted, against
    the oracle's conversion of the oracle's propagation; the intensity also in place; and the complex output again once the
    option is switched off."""
    op, shape = case
    ny, nx = shape
    px, py, lam = 4e-6, 5e-6, 633e-9
    u1 = _rand_field(shape, 17 + nx % 13)
    z = max(nx, ny) * px * px / lam * 0.35
    plan = api.cwo_plan(nx, ny, px, lam)
    plan.set_pitch_xy(px, py)
    if op == "asm":
        call, ref = api.cwo_asm, oracle.asm(u1, px, py, lam, z)
    elif op == "asm_pad2x":
        plan.set_option(api.CWO_OPT_ASM_PAD2X, 1)
        call, ref = api.cwo_asm, oracle.asm_pad2x(u1, px, py, lam, z)
    elif op == "fresnel":
        call, ref = api.cwo_fresnel_conv, oracle.fresnel_conv(u1, px, py, lam, z)
    elif op == "fourier":
        call, ref = api.cwo_fresnel_fourier, oracle.fresnel_fourier(u1, px, py, lam, z)
    else:
        p1, off = (1.3 * px, 0.8 * py), (11.5 * px, -20.25 * py)
        plan.set_dst_pitch_xy(*p1); plan.set_offset(*off)
        call, ref = api.cwo_fresnel_shifted, oracle.fresnel_shifted(u1, (px, py), p1, lam, z, (0.0, 0.0), off)
    d1 = torch.from_numpy(u1).cuda()
    peak = np.abs(ref).max()
    outs = {}
    for mode, conv in ((api.CWO_OUT_INTENSITY, oracle.intensity), (api.CWO_OUT_AMPLITUDE, oracle.amplitude),
                       (api.CWO_OUT_RE, oracle.re), (api.CWO_OUT_IM, oracle.im), (api.CWO_OUT_PHASE, oracle.phase)):
        plan.set_option(api.CWO_OPT_OUT_REAL, mode)
        out = torch.full((ny, nx), -7.0, dtype=torch.float32, device="cuda")
        call(plan, d1, out, z)
        torch.cuda.synchronize()
        got = out.cpu().numpy().astype(np.float64)
        outs[mode] = out
        want = conv(ref)
        what = "%s %s mode %d" % (op, shape, mode)
        if mode == api.CWO_OUT_INTENSITY:
            _assert_intensity(got, want, what)
        elif mode == api.CWO_OUT_PHASE:
            # the phase is ill-conditioned where |u2| is small (an error e moves it by e/|u2|): compare the phasors, weighted
            # by the amplitude, at the propagation bars; and the range of Eq.(25)
            assert got.min() >= -np.pi - 1e-6 and got.max() <= np.pi + 1e-6
            d = np.abs(ref) * np.abs(np.exp(1j * got) - np.exp(1j * want))
            assert np.linalg.norm(d) / np.linalg.norm(ref) <= REL_L2 and d.max() <= MAX_ABS * peak, what
        else:
            # |u|, Re, Im carry the error of u itself: the propagation bars, relative to the field's norm and peak
            d = np.abs(got - want)
            assert np.linalg.norm(d) / np.linalg.norm(ref) <= REL_L2 and d.max() <= MAX_ABS * peak, what
    assert torch.equal(d1.cpu(), torch.from_numpy(u1))                    # the input is untouched
    # in place: the real field occupies the first half of u1's bytes
    plan.set_option(api.CWO_OPT_OUT_REAL, api.CWO_OUT_INTENSITY)
    with pytest.raises(TypeError):
        call(plan, d1, d1, z)                                             # the binding wants a float32 tensor for u2
    inplace = d1.view(torch.float32).view(-1)[: nx * ny].view(ny, nx)
    call(plan, d1, inplace, z)
    torch.cuda.synchronize()
    assert torch.equal(inplace, outs[api.CWO_OUT_INTENSITY])
    # option off again: complex output at the usual bar
    plan.set_option(api.CWO_OPT_OUT_REAL, api.CWO_OUT_COMPLEX)
    d1 = torch.from_numpy(u1).cuda(); d2 = torch.empty_like(d1)
    call(plan, d1, d2, z)
    torch.cuda.synchronize()
    got = d2.cpu().numpy().astype(np.complex128)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= REL_L2
    with pytest.raises(api.CwoError):
        plan.set_option(api.CWO_OPT_OUT_REAL, 6)
