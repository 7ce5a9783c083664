"""Error behaviour of the C-ABI on a GPU box (include/lartpc.h states it per entry point): wrong call order, buffers that
are too small, parameters out of range come back as negative codes through the binding's LartpcError, never as a fault."""
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


def _code(exc):
    return int(str(exc.value).rsplit("(", 1)[1].rstrip(")"))


def test_charge_path_errors(lartpc):
    import torch
    wl = W.make_config(0)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    dr = sim.drift(seg, ne)
    # the truth pass needs the plan of S3 and the hits of S6
    hp = torch.zeros(4, dtype=torch.int32, device="cuda")
    fake_hits = {"counters": torch.zeros(4, dtype=torch.int64, device="cuda"),
                 "_struct": lartpc.Hits(4, hp.data_ptr(), hp.data_ptr(), hp.data_ptr(), None, None, None)}
    pm_fake = {k: torch.zeros(len(wl.segments["xs"]), dtype=torch.int32, device="cuda") for k in lartpc._PIX_I32}
    pm_fake["offsets"] = torch.zeros(len(wl.segments["xs"]) + 1, dtype=torch.int64, device="cuda")
    pm_fake["_struct"] = lartpc.Pixmap(**{k: v.data_ptr() for k, v in pm_fake.items()})
    with pytest.raises(lartpc.LartpcError) as e:
        sim.hit_truth(dr, pm_fake, fake_hits, 1, k_max=2)
    assert _code(e) == -7                                            # LARTPC_ERR_ORDER
    with pytest.raises(lartpc.LartpcError) as e:
        sim.set_truncation_compensation(-1.0)
    assert _code(e) == -1                                            # LARTPC_ERR_BAD_ARGUMENT
    with pytest.raises(lartpc.LartpcError) as e:
        sim.set_truncation_compensation(1e-3)
    assert _code(e) == -1
    pm, _ = sim.pixels_from_segments(seg, dr)
    wf = sim.sum_pixel_signals(sim.induced_current(dr, pm))
    hits = sim.electronics(wf, 1)
    with pytest.raises(lartpc.LartpcError) as e:
        sim.hit_truth(dr, pm, hits, k_max=0)
    assert _code(e) == -1
    # a workspace that is too small for one TPC is a capacity error, not a fault
    with pytest.raises(lartpc.LartpcError) as e:
        sim.run_spill(seg, 1, 4096, workspace=torch.empty(1 << 12, dtype=torch.uint8, device="cuda"))
    assert _code(e) in (-2, -1)
    sim.close()


def test_light_errors(lartpc):
    import torch
    wl = W.make_config(0)
    ls = W.light_setup(wl, n_det=4)
    for bad in (dict(n_ticks=0), dict(lut_m=0), dict(tick_us=0.0), dict(n_det=0), dict(tau_slow_us=-1.0)):
        p = dict(ls.params, **bad)
        with pytest.raises(lartpc.LartpcError) as e:
            lartpc.LightSim(p, ls.eff[:max(p["n_det"], 1)], ls.gain[:max(p["n_det"], 1)], ls.vis[:max(p["n_det"], 1)],
                            ls.tprof[:max(p["n_det"], 1)], ls.resp)
        assert "tables do not" in str(e.value) or _code(e) == -1
    light = lartpc.LightSim(ls.params, ls.eff, ls.gain, ls.vis, ls.tprof, ls.resp)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    with pytest.raises(lartpc.LartpcError) as e:
        light.run(seg, ne, 1, workspace=torch.empty(256, dtype=torch.uint8, device="cuda"))
    assert _code(e) == -2                                            # LARTPC_ERR_CAPACITY
    assert light.workspace_bytes(len(wl.segments["xs"])) > 0
    # a 1 ns tick makes the scintillation kernel 8 001 taps long: still inside the shared-memory budget
    p = dict(ls.params, tick_us=0.001, n_ticks=2048, lut_m=16)
    l2 = lartpc.LightSim(p, ls.eff, ls.gain, ls.vis, ls.tprof, ls.resp)
    v = l2.run(seg, ne, 1)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(v).all())
    l2.close()
    light.close()
    sim.close()
