"""cwo_scale255_static: Scale (Eq.(21)) for callers that are not allowed to allocate device memory.

cwo_scale255 needs a plan, and cwo_plan() gets its tables from cudaMalloc.  A caller that works while a CUDA graph is
being captured elsewhere in the process, that lives inside a host owning all device memory through its own pool, or
that cannot take cudaMalloc's device-wide synchronisation has no way to make one.  cwo_scale255_static takes no plan:
its scratch is a fixed 256 KiB array inside libcwo.so, which limits it to 2**28 floats per call.  These tests compare
it with the plan path (it must give the same numbers: the map is the same kernel, and min / max do not depend on the
order of reduction) and with the oracle, on calls issued back to back -- the array is shared by every call and keeps
what the previous call left, so the second call must not be disturbed by the first.

This file is collected last on purpose (pytest -x stops at the first failure); it passes alone in a fresh process,
where its first call also performs the per-device set-up, and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from test_gpu_parity import api   # noqa: E402,F401

TOL = 255 * 4e-7 * 8          # the bound test_gpu_outputs.py::test_scale255_matches_oracle uses
CHUNK = 8192                  # floats per scratch slot (scale_static.cu SS_CHUNK)


def _plan_path(api, d):
    plan = api.cwo_plan(256, 256, 4e-6, 633e-9)
    ref = torch.empty_like(d)
    api.cwo_scale255(plan, d, ref)
    torch.cuda.synchronize()
    return ref.cpu().numpy()


def test_two_calls_in_a_row_match_the_plan_path_and_the_oracle(api, oracle):
    r = np.random.default_rng(2024)
    # first call: six chunk slots and a tail that is not a multiple of four, values in about [-3, 600]
    a1 = (r.standard_normal(5 * CHUNK + 4099) ** 2 * 37.0 - 3.0).astype(np.float32)
    # second call: fewer slots and a much narrower range -- any slot left over from the first call that leaked into
    # this one would move its minimum and maximum
    a2 = r.uniform(10.0, 11.0, CHUNK + 7).astype(np.float32)
    d1, d2 = torch.from_numpy(a1).cuda(), torch.from_numpy(a2).cuda()
    o1, o2 = torch.empty_like(d1), torch.empty_like(d2)
    torch.cuda.synchronize()
    api.cwo_scale255_static(d1, o1)           # in a fresh process this call also resolves the array's device address
    api.cwo_scale255_static(d2, o2)           # straight after it on the same stream, no synchronisation in between
    torch.cuda.synchronize()
    for a, d, o in ((a1, d1, o1), (a2, d2, o2)):
        got, ref = o.cpu().numpy(), _plan_path(api, d)
        assert np.abs(got - ref).max() <= TOL
        assert np.array_equal(got, ref)
        assert np.abs(got - oracle.scale255(a.astype(np.float64))).max() <= TOL
        assert got.min() == 0.0 and got.max() == 255.0
    # the same pair again in the other order and in place (out == in)
    api.cwo_scale255_static(d2, d2)
    api.cwo_scale255_static(d1, d1)
    torch.cuda.synchronize()
    assert np.array_equal(d1.cpu().numpy(), o1.cpu().numpy()) and np.array_equal(d2.cpu().numpy(), o2.cpu().numpy())


@pytest.mark.parametrize("n", [1, 5, CHUNK, CHUNK + 1, 4096 * 4096])
def test_sizes_from_one_float_to_many_chunks(api, n):
    a = (np.random.default_rng(n).standard_normal(n) * 5.0 + 1.0).astype(np.float32)
    d = torch.from_numpy(a).cuda()
    o = torch.empty_like(d)
    api.cwo_scale255_static(d, o)
    api.cwo_scale255_static(d, o)
    torch.cuda.synchronize()
    ref = _plan_path(api, d)
    assert np.abs(o.cpu().numpy() - ref).max() <= TOL and np.array_equal(o.cpu().numpy(), ref)


def test_no_device_memory_is_taken_by_a_call(api):
    d = torch.rand(3 * CHUNK + 5, device="cuda")
    o = torch.empty_like(d)
    api.cwo_scale255_static(d, o)             # set-up and module load, if this is the first call of the process
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    reserved0 = torch.cuda.memory_reserved()
    api.cwo_scale255_static(d, o)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0 and torch.cuda.memory_reserved() == reserved0


def test_the_largest_size_and_the_refusal_beyond_it(api):
    nmax = api.CWO_SCALE255_STATIC_MAX_N
    # one float more than the scratch has slots for: refused before anything is enqueued, pointers are not touched
    d = torch.rand(16, device="cuda")
    err = ctypes.c_int(-1)
    rc = api.lib().cwo_scale255_static(d.data_ptr(), d.data_ptr(), nmax + 1, None, ctypes.byref(err))
    assert rc == api.CWO_ELIMIT and err.value == 0
    assert b"CWO_SCALE255_STATIC_MAX_N" in api.lib().cwo_strerror(rc)
    assert api.lib().cwo_scale255_static(d.data_ptr(), d.data_ptr(), 0, None, None) == api.CWO_EINVAL
    assert api.lib().cwo_scale255_static(d.data_ptr() + 4, d.data_ptr(), 4, None, None) == api.CWO_EINVAL
    # exactly the limit (1 GiB of floats, every slot of the array in use), against the plan path
    big = torch.rand(nmax, device="cuda")
    big[12345] = -2.0; big[nmax - 3] = 7.0
    out = torch.empty_like(big)
    api.cwo_scale255_static(big, out)
    torch.cuda.synchronize()
    plan = api.cwo_plan(256, 256, 4e-6, 633e-9)
    api.cwo_scale255(plan, big, big)
    torch.cuda.synchronize()
    assert torch.equal(out, big)
    assert float(out[12345]) == 0.0 and float(out[nmax - 3]) == 255.0
