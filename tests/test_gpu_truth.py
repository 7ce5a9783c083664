"""GPU parity of lartpc_hit_truth (reading D26) against oracle O7: for every hit checked, the
share q_{h,s} of every segment the GPU lists, the hit's total and the membership of the top-k list."""
import numpy as np
import pytest

import oracle
from paper_2212_09807_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lartpc():
    from paper_2212_09807_b200 import lartpc as mod
    mod.load_library()
    return mod


def _run(lartpc, wl, k_max, mode="tensor"):
    import torch
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response=mode)
    if wl.disabled_pixels is not None:
        sim.set_disabled_pixels(wl.disabled_pixels)
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    dr = sim.drift(seg, ne)
    pm, _ = sim.pixels_from_segments(seg, dr)
    wf = sim.sum_pixel_signals(sim.induced_current(dr, pm))
    hits = sim.electronics(wf, wl.seed)
    n = int(hits["counters"][0].item())
    tr = sim.hit_truth(dr, pm, hits, n, k_max=k_max)
    torch.cuda.synchronize()
    out = dict(pixel=hits["hit_pixel"][:n].cpu().numpy(), tick=hits["hit_tick"][:n].cpu().numpy(),
               adc=hits["hit_adc"][:n].cpu().numpy(), **{k: v.cpu().numpy() for k, v in tr.items()})
    sim.close()
    return out


def _check_truth(wl, got, pixel_ids, k_max):
    """Oracle O7 on the listed pixels (global ids); compares every hit of those pixels."""
    _, ne = oracle.quench(wl.params, wl.segments)
    dr = oracle.drift(wl.params, wl.tpcs, wl.segments, ne)
    pm = oracle.pixmap(wl.params, wl.tpcs, wl.segments, dr)
    n_checked = n_entries = 0
    worst = 0.0
    for pid in pixel_ids:
        ti = [i for i, t in enumerate(wl.tpcs) if t["first_pixel_id"] <= pid < t["first_pixel_id"] + t["nx"] * t["ny"]][0]
        t = wl.tpcs[ti]
        rel = pid - t["first_pixel_id"]
        ix, iy = rel % t["nx"], rel // t["nx"]
        # candidates: segments of this TPC whose O3 rectangle holds the pixel (beyond it a segment carries < 2e-6 of its charge)
        sel = np.nonzero((dr["tpc"] == ti) & (pm["ix0"] <= ix) & (ix <= pm["ix1"]) & (pm["iy0"] <= iy) & (iy <= pm["iy1"]))[0]
        waves, _ = oracle.pixel_currents(wl.params, wl.tpcs, wl.lut, dr, pm, ti, [ix], [iy])
        hp, ht, ha, _ = oracle.electronics(wl.params, wl.seed, [pid], waves)
        mine = np.nonzero(got["pixel"] == pid)[0]
        if len(ht) != len(mine) or not np.array_equal(got["tick"][mine], ht):
            continue                                            # a near miss moved this pixel's chain: windows differ
        sw = oracle.segment_currents(wl.params, wl.tpcs, wl.lut, dr, pm, ti, ix, iy, sel)
        n0, share = oracle.hit_truth(wl.params, ht, sw)
        for k, h in enumerate(mine):
            q_o = share[k].sum()
            tol_q = max(1e-4 * np.abs(share[k]).sum(), 1.0)      # shares of both signs: the tolerance follows the gross sum
            assert abs(got["q_signal"][h] - q_o) <= tol_q, (pid, k, got["q_signal"][h], q_o)
            segs, fr = got["seg"][h], got["frac"][h]
            used = segs >= 0
            assert len(set(segs[used].tolist())) == used.sum()
            order = np.argsort(-np.abs(share[k]), kind="stable")
            kth = np.abs(share[k][order[min(k_max, len(sel)) - 1]]) if len(sel) else 0.0
            for s_id, f in zip(segs[used], fr[used]):
                pos = np.nonzero(sel == s_id)[0]
                assert len(pos) == 1, "GPU lists a segment outside the oracle's candidates"
                q_s = share[k][pos[0]]
                tol = max(1e-4 * abs(q_s), 1.0)
                assert abs(f * got["q_signal"][h] - q_s) <= tol + abs(f) * tol_q, (pid, k, s_id, f * got["q_signal"][h], q_s)
                worst = max(worst, abs(f * got["q_signal"][h] - q_s) / (tol + abs(f) * tol_q))
                assert abs(q_s) >= kth - 2.0                    # it belongs to the k largest (ties within the tolerance)
                n_entries += 1
            # every clearly larger share of the oracle is listed, in decreasing order
            must = [int(sel[i]) for i in order[:k_max] if abs(share[k][i]) > kth + 2.0 and abs(share[k][i]) > 2.0]
            assert set(must) <= set(segs[used].tolist()), (pid, k)
            mags = np.abs(fr[used])
            assert np.all(mags[:-1] >= mags[1:] - 1e-6)
            assert got["n_contrib"][h] >= int((np.abs(share[k]) > 1.0).sum())
            if used.sum() == got["n_contrib"][h]:
                assert fr[used].sum() == pytest.approx(1.0, abs=1e-4)
            n_checked += 1
    return n_checked, n_entries, worst


@pytest.mark.parametrize("variant", ["plain", "periodic_reset", "low_threshold"])
def test_hit_truth_config0(lartpc, variant):
    """BASELINE configs[0] (one MIP track, no noise): every hit of every pixel.  Variants move the windows: a periodic
    reset (window starts at a reset tick) and a low threshold (several hits per pixel, windows back to back)."""
    wl = W.make_config(0)
    if variant == "periodic_reset":
        wl.params.update(periodic_reset_ticks=97)
    elif variant == "low_threshold":
        wl.params.update(threshold_e=3000.0)
    got = _run(lartpc, wl, k_max=6)
    assert len(got["pixel"]) > 20
    n, ne, worst = _check_truth(wl, got, sorted(set(got["pixel"].tolist())), 6)
    assert n == len(got["pixel"]) and ne > 3 * n
    print("truth %s: %d hits, %d (hit, segment) shares checked, worst error / tolerance %.3f" % (variant, n, ne, worst))


def test_hit_truth_zero_sigma_and_edges(lartpc):
    """Segments at the anode (sigma = 0: one-hot weights, float64 bin decisions) and at the plane edge (source pixels in
    the margin outside the plane)."""
    p = W.default_params(n_readout_ticks=900)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, 10.0, 16, 16, 0)]
    pitch = p["pixel_pitch_cm"]
    parts = [
        W.line_segments([3.3 * pitch, 4.2 * pitch, 0.0], [6.1 * pitch, 5.9 * pitch, 0.0], 0.1, 0.5, W._mip(2.1)),
        W.line_segments([0.05 * pitch, 7.0 * pitch, 4.0], [2.0 * pitch, 7.7 * pitch, 4.3], 0.1, 0.0, W._mip(2.1)),
        W.line_segments([14.0 * pitch, 15.95 * pitch, 2.0], [15.9 * pitch, 15.6 * pitch, 2.5], 0.1, 0.0, W._mip(2.1)),
        W.line_segments([4.0 * pitch, 4.9 * pitch, 1.0], [5.5 * pitch, 5.2 * pitch, 1.2], 0.05, 0.5, W._mip(4.0)),   # overlaps the anode track in time
    ]
    wl = W.Workload("truth-edges", 7, p, tpcs, W._concat(parts), W.pad_response_lut(p))
    got = _run(lartpc, wl, k_max=8)
    assert len(got["pixel"]) > 8
    n, ne, worst = _check_truth(wl, got, sorted(set(got["pixel"].tolist())), 8)
    assert n == len(got["pixel"])
    print("truth edges: %d hits, %d shares checked, worst error / tolerance %.3f" % (n, ne, worst))


def test_hit_truth_config2_sample(lartpc):
    """BASELINE configs[2] (1e5 segments, showers, Birks, noise on): the hits of the 3 busiest and 3 random hit pixels
    per TPC; pixels whose GPU hit ticks differ from the oracle's (a near miss) are left out, at least 30 must remain."""
    wl = W.make_config(2)
    got = _run(lartpc, wl, k_max=4)
    rng = np.random.Generator(np.random.PCG64(5))
    picks = []
    for t in wl.tpcs:
        m = (got["pixel"] >= t["first_pixel_id"]) & (got["pixel"] < t["first_pixel_id"] + t["nx"] * t["ny"])
        ids, cnt = np.unique(got["pixel"][m], return_counts=True)
        if len(ids) == 0:
            continue
        picks += ids[np.argsort(cnt)[-3:]].tolist() + rng.choice(ids, size=min(3, len(ids)), replace=False).tolist()
    n, ne, worst = _check_truth(wl, got, sorted(set(picks)), 4)
    assert n >= 30
    print("truth configs[2]: %d hits of %d pixels, %d shares checked, worst error / tolerance %.3f" % (n, len(set(picks)), ne, worst))
