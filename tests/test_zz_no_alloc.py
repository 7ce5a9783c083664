"""lartpc_electronics_static (include/lartpc.h): S6 with its scratch in a fixed file-scope device array, for callers that
must not allocate.  Its output is compared with lartpc_electronics' on the same waveforms: S6 is integer work on both sides
(same kernels, same order), so the bar is the one the parity tests hold integer output to: bit-exact (hit pixel / tick / ADC,
counters, hits per pixel; q_pixel is the same float32 sum, compared exactly too).  The scratch keeps the last call's
contents, so the calls follow one another on purpose: same input twice, another seed, then a smaller workload of another sim.

This file is collected last (pytest --collect-only): the suite runs with pytest -x and a failure here must not hide the
parity tests.  It passes alone in a fresh process and after the others (nothing here depends on what ran before)."""
import ctypes as C

import numpy as np
import pytest

from paper_2212_09807_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lartpc():
    from paper_2212_09807_b200 import lartpc as mod
    mod.load_library()
    return mod


def _waveforms(sim, wl):
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    dr = sim.drift(seg, ne)
    pm, _ = sim.pixels_from_segments(seg, dr)
    sig = sim.induced_current(dr, pm)
    return sim.sum_pixel_signals(sig), (seg, ne, dr, pm, sig)


def _as_numpy(h, na):
    n = int(h["counters"][0].item())
    return dict(counters=h["counters"].cpu().numpy().copy(), pixel=h["hit_pixel"][:n].cpu().numpy().copy(),
                tick=h["hit_tick"][:n].cpu().numpy().copy(), adc=h["hit_adc"][:n].cpu().numpy().copy(),
                per_pixel=h["hits_per_pixel"][:na].cpu().numpy().copy(), q=h["q_pixel"][:na].cpu().numpy().copy())


def _same(a, b):
    for k in a:
        assert np.array_equal(a[k], b[k]), k
    assert a["counters"][0] > 0


def test_static_scratch_electronics_matches_the_allocating_path(lartpc):
    import torch
    wl = W.make_config(1)                                             # cosmics, reset and uncorrelated noise on
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    wf, keep = _waveforms(sim, wl)
    na = int(wf["_struct"].n_active)
    assert 0 < na <= 65536
    ref = _as_numpy(sim.electronics(wf, wl.seed), na)
    ref2 = _as_numpy(sim.electronics(wf, wl.seed + 1), na)
    assert not np.array_equal(ref["adc"], ref2["adc"]) or not np.array_equal(ref["tick"], ref2["tick"])   # the noise is on
    # two calls in a row on the same input, then another seed: each equal to the existing path
    h1 = sim.electronics_static(wf, wl.seed)
    h2 = sim.electronics_static(wf, wl.seed)
    torch.cuda.synchronize()
    _same(_as_numpy(h1, na), ref)
    _same(_as_numpy(h2, na), ref)
    _same(_as_numpy(sim.electronics_static(wf, wl.seed + 1), na), ref2)
    # the same call again straight through the C-ABI into the buffers of h2: the device's free memory does not move
    lib = lartpc.load_library()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(2):
        rc = lib.lartpc_electronics_static(sim.handle, C.byref(wf["_struct"]), C.c_uint64(wl.seed), C.byref(h2["_struct"]),
                                           C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == 0
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    _same(_as_numpy(h2, na), ref)
    # a smaller workload on another sim, over whatever the calls above left in the scratch
    wl0 = W.make_config(0)
    sim0 = lartpc.Sim(wl0.params, wl0.tpcs, wl0.lut)
    wf0, keep0 = _waveforms(sim0, wl0)
    na0 = int(wf0["_struct"].n_active)
    ref0 = _as_numpy(sim0.electronics(wf0, wl0.seed), na0)
    _same(_as_numpy(sim0.electronics_static(wf0, wl0.seed), na0), ref0)
    _same(_as_numpy(sim0.electronics_static(wf0, wl0.seed), na0), ref0)
    # and the larger one once more
    _same(_as_numpy(sim.electronics_static(wf, wl.seed), na), ref)
    sim0.close()
    sim.close()


def test_static_scratch_limit_is_an_error(lartpc):
    """More active pixels (or hit slots) than the fixed scratch holds: a clear error, nothing launched."""
    import torch
    wl = W.make_config(0)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    wf, keep = _waveforms(sim, wl)
    na = int(wf["_struct"].n_active)
    good = sim.electronics_static(wf, wl.seed)
    torch.cuda.synchronize()
    before = _as_numpy(good, na)
    lib = lartpc.load_library()
    big = type(wf["_struct"]).from_buffer_copy(wf["_struct"])
    for n_active in (65536 + 1, 2097152 // int(wl.params["max_hits_per_pixel"]) + 1, 1 << 40):
        big.n_active = n_active
        rc = lib.lartpc_electronics_static(sim.handle, C.byref(big), C.c_uint64(wl.seed), C.byref(good["_struct"]),
                                           C.c_void_p(torch.cuda.current_stream().cuda_stream))
        assert rc == -8
        msg = lib.lartpc_strerror(rc).decode()
        assert "lartpc_electronics_static" in msg and "LARTPC_STATIC_MAX_PIXELS" in msg
    big.n_active = 65536                                              # the limit itself is accepted by the size check
    torch.cuda.synchronize()
    _same(_as_numpy(good, na), before)                                # the refused calls wrote nothing
    with pytest.raises(lartpc.LartpcError):
        big.n_active = 65537
        lartpc._check(lib.lartpc_electronics_static(sim.handle, C.byref(big), C.c_uint64(0), C.byref(good["_struct"]), None),
                      "lartpc_electronics_static")
    sim.close()
