"""Bit-exact repeatability of every call (compute-sanitizer is not available on this pool: a data race in the
exchange / barrier / TMA protocols of the kernels would show up as run-to-run differences).  No kernel accumulates in
floating point through atomics, so identical inputs must give identical bits, back to back and under load."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from paper_1107_5578_b200 import workloads as W   # noqa: E402
from test_gpu_parity import _dev, _rand, api   # noqa: E402,F401

REPS = 12


def _same(ref, t, what, i):
    assert torch.equal(ref.view(torch.uint8), t.view(torch.uint8)), "%s: run %d differs from run 0" % (what, i)


@pytest.mark.parametrize("n", [256, 2048, 4096, 8192])
def test_asm_is_bit_repeatable(api, n):
    cfg = W.CONFIGS["c3"]
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    d1 = _dev(_rand((n, n), n)); ref = None
    outs = [torch.empty_like(d1) for _ in range(3)]
    for i in range(REPS):
        o = outs[i % 3]
        o.zero_()
        api.cwo_asm(plan, d1, o, 0.1)
        if i == 0:
            torch.cuda.synchronize(); ref = o.clone()
        else:
            _same(ref, o, "asm %d" % n, i)


@pytest.mark.parametrize("n,mode", [(512, -1), (2048, 0), (2048, 1), (4096, -1), (8192, -1)])
def test_fresnel_forms_are_bit_repeatable(api, n, mode):
    cfg = W.CONFIGS["c5"]
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    plan.set_fresnel_gather(mode)
    plan.set_dst_pitch_xy(1.5 * cfg.pitch, 0.8 * cfg.pitch); plan.set_offset(1e-4, -2e-4)
    d1 = _dev(_rand((n, n), n + 1))
    reps = REPS if n < 8192 else 6
    for call in (api.cwo_fresnel_conv, api.cwo_fresnel_shifted, api.cwo_fresnel_fourier):
        ref = None
        outs = [torch.empty_like(d1) for _ in range(2)]
        for i in range(reps):
            o = outs[i % 2]
            o.zero_()
            call(plan, d1, o, 0.3 * n / 8192)
            if i == 0:
                torch.cuda.synchronize(); ref = o.clone()
            else:
                _same(ref, o, "%s %d" % (call.__name__, n), i)


def test_stack_gs_and_outputs_are_bit_repeatable(api):
    n = 1024
    cfg = W.CONFIGS["c4"].scaled(n)
    plan = api.cwo_plan(n, n, cfg.pitch, cfg.lam)
    d1 = _dev(W.make_field(cfg))
    zs = list(cfg.zs[:20])
    st = torch.empty((20, n, n), dtype=torch.complex64, device="cuda")
    ref = None
    for i in range(6):
        st.zero_()
        api.cwo_propagate_stack(plan, d1, zs, st)
        if i == 0:
            torch.cuda.synchronize(); ref = st.clone()
        else:
            _same(ref, st, "stack", i)
    amp_src, amp_dst, phi0 = W.gs_inputs((n, n), 5)
    for method in (0, 1):
        plan.set_option(api.CWO_OPT_GS_METHOD, method)
        ref = None
        for i in range(6):
            ph = _dev(phi0.copy())
            api.cwo_gs(plan, _dev(amp_src), _dev(amp_dst), 0.05, 3, ph)
            if i == 0:
                torch.cuda.synchronize(); ref = ph.clone()
            else:
                _same(ref, ph, "gs method %d" % method, i)
    pts = torch.from_numpy(np.random.default_rng(1).uniform(-1e-3, 1e-3, (300, 4)) + np.array([0, 0, 0.2, 1.0])).cuda()
    holo = torch.empty((n, n), dtype=torch.float32, device="cuda"); s8 = torch.empty_like(holo)
    ref = ref8 = None
    for i in range(6):
        api.cwo_pls_cgh(plan, pts, holo); api.cwo_scale255(plan, holo, s8)
        if i == 0:
            torch.cuda.synchronize(); ref = holo.clone(); ref8 = s8.clone()
        else:
            _same(ref, holo, "pls", i); _same(ref8, s8, "scale255", i)
