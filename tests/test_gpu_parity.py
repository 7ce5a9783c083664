"""Parity of the CUDA path (through the C-ABI) with the fp64 oracle, element by element, on seeded inputs.

Tolerances are BASELINE.json north_star's: pixel mapping bit-exact; per-pixel integrated charge within
relative 1e-4 (absolute 1 e-); >= 99.9 % of hits identical in (pixel, tick, adc), the rest off by <= 1 tick
or 1 count.  Float32 stage outputs (S1, S2) are held to 2e-6 relative (a few float32 ulp).
"""
import numpy as np
import pytest

import oracle
from paper_2212_09807_b200 import workloads as W

from gpu_helpers import compare_hits, dense_waves, run_staged

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lartpc():
    from paper_2212_09807_b200 import lartpc as L
    L.load_library()
    return L


def _oracle_stages(wl):
    dedx, ne = oracle.quench(wl.params, wl.segments)
    dr = oracle.drift(wl.params, wl.tpcs, wl.segments, ne)
    pm = oracle.pixmap(wl.params, wl.tpcs, wl.segments, dr)
    return dedx, ne, dr, pm


def _check_segment_stages(res, wl):
    dedx, ne, dr, pm = _oracle_stages(wl)
    assert np.allclose(res["dEdx"], dedx, rtol=2e-6, atol=0)
    assert np.allclose(res["n_e"], ne, rtol=2e-6, atol=1e-3)
    g = res["drift"]
    assert np.array_equal(g["tpc"], dr["tpc"])
    assert np.allclose(g["q_anode"], dr["q_a"], rtol=2e-6, atol=1e-3)
    assert np.allclose(g["sigma_T"], dr["sigma_T"], rtol=2e-7, atol=0)
    assert np.allclose(g["sigma_t"], dr["sigma_t"], rtol=2e-7, atol=0)
    for a, b in (("u_s", "u_s"), ("v_s", "v_s"), ("u_e", "u_e"), ("v_e", "v_e"), ("T_s", "T_s"), ("T_e", "T_e")):
        assert np.array_equal(g[a], dr[b]), a                      # float64, same operations: bit-exact
    gp = res["pixmap"]
    for k in ("a_lo", "a_hi", "b_lo", "b_hi", "ix0", "ix1", "iy0", "iy1", "jt0", "jt1", "npix", "n_samples"):
        assert np.array_equal(gp[k], pm[k]), k                     # pixel mapping: bit-exact
    assert np.array_equal(gp["offsets"], pm["offsets"])
    info = res["info"]
    assert info.max_npix == pm["npix"].max()
    assert info.total_npix == pm["offsets"][-1]
    act = pm["npix"] > 0
    assert info.n_active_segments == act.sum()
    if act.any():
        assert info.max_ticks == (pm["jt1"] - pm["jt0"] + 1)[act].max() + wl.params["lut_ticks"] - 1
    return dr, pm


def _check_currents(res, wl, dr, pm, max_pixels=None, seed=0):
    """Waveforms and Q_p of (a sample of) the active pixels against O4/O5."""
    nt = wl.params["n_readout_ticks"]
    dense = dense_waves(res, nt)
    gpu_ids = res["waveforms"]["pixel_id"][:res["n_active"]]
    # active set = union of the O3 rectangles
    ids = []
    for ti, t in enumerate(wl.tpcs):
        ix, iy = oracle.active_pixels(wl.tpcs, pm, dr, ti)
        ids.append(t["first_pixel_id"] + iy.astype(np.int64) * t["nx"] + ix)
    ids = np.concatenate(ids)
    assert np.array_equal(np.sort(ids), gpu_ids)
    rng = np.random.Generator(np.random.PCG64(seed))
    worst_q, worst_w = 0.0, 0.0
    for ti, t in enumerate(wl.tpcs):
        sel = np.nonzero((gpu_ids >= t["first_pixel_id"]) & (gpu_ids < t["first_pixel_id"] + t["nx"] * t["ny"]))[0]
        if len(sel) == 0:
            continue
        if max_pixels is not None and len(sel) > max_pixels:
            # the pixels carrying the most charge plus a random sample of the rest
            q = np.abs(dense[sel]).sum(axis=1)
            top = sel[np.argsort(q)[-max_pixels // 2:]]
            rest = rng.choice(sel, size=max_pixels // 2, replace=False)
            sel = np.unique(np.concatenate([top, rest]))
        rel = gpu_ids[sel] - t["first_pixel_id"]
        waves, qp = oracle.pixel_currents(wl.params, wl.tpcs, wl.lut, dr, pm, ti, rel % t["nx"], rel // t["nx"])
        gq = dense[sel].sum(axis=1)
        tol = np.maximum(1e-4 * np.abs(qp), 1.0)
        assert np.all(np.abs(gq - qp) <= tol), (np.abs(gq - qp) / tol).max()
        worst_q = max(worst_q, (np.abs(gq - qp) / tol).max())
        # sample by sample: 1e-4 of the pixel's peak current plus 0.02 e- (float32 accumulation of ~1e4 terms)
        peak = np.abs(waves).max(axis=1, keepdims=True)
        err = np.abs(dense[sel] - waves)
        assert np.all(err <= 1e-4 * peak + 0.02), (err / (1e-4 * peak + 0.02)).max()
        worst_w = max(worst_w, (err / (1e-4 * peak + 0.02)).max())
        # Q_p reported by S6 is the same sum
        assert np.allclose(res["hits"]["q_pixel"][sel], gq, rtol=1e-5, atol=0.05)
    print("currents vs oracle: worst |dQ| / tol = %.3f, worst sample error / tol = %.3f" % (worst_q, worst_w))
    return worst_q, worst_w


def _check_hits(res, wl, dr, pm, seed):
    """S6 on the oracle's own currents of every active pixel (full chain parity)."""
    r = oracle.run_chain(wl, seed=seed)
    h = res["hits"]
    n = int(h["counters"][0])
    gpu = (h["hit_pixel"][:n], h["hit_tick"][:n], h["hit_adc"][:n])
    frac, near, ng, no = compare_hits(gpu, (r["hit_pixel"], r["hit_tick"], r["hit_adc"]))
    assert no > 0
    assert frac >= 0.999 and near, (frac, near, ng, no)
    assert ng == no
    # sorted by (pixel, tick)
    key = gpu[0].astype(np.int64) * (1 << 20) + gpu[1]
    assert np.all(np.diff(key) > 0)
    return frac


MODES = ["tensor", "ffma"]          # both S4 response paths are held to the same bar


@pytest.mark.parametrize("mode", MODES)
def test_config0_full_chain(lartpc, mode):
    """BASELINE configs[0]: 100 segments of one MIP track, every stage and every active pixel."""
    wl = W.make_config(0)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response=mode)
    assert sim.response_mode == mode
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm)
    _check_hits(res, wl, dr, pm, wl.seed)
    sim.close()


@pytest.mark.parametrize("seed", [7, 8, 9])
def test_config0_other_tracks(lartpc, seed):
    wl = W.make_config(0, seed=seed)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm)
    _check_hits(res, wl, dr, pm, wl.seed)
    sim.close()


def test_run_spill_matches_staged(lartpc):
    """lartpc_run_spill gives the same hit list as the staged calls (same kernels, bit for bit)."""
    wl = W.make_config(0)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, wl)
    seg = sim.upload_segments(wl.segments)
    hits, st = sim.run_spill(seg, wl.seed, hit_capacity=4096)
    n = int(res["hits"]["counters"][0])
    assert st.n_hits == n and st.n_hits_total == n and st.n_hits_dropped == 0
    assert st.n_tiles == res["info"].n_tiles and st.n_active_pixels == res["n_active"]
    got = lartpc.hits_to_numpy(hits)
    for a, k in zip(got, ("hit_pixel", "hit_tick", "hit_adc")):
        assert np.array_equal(a, res["hits"][k][:n])
    sim.close()


@pytest.mark.parametrize("mode", MODES)
def test_config1_sampled_pixels(lartpc, mode):
    """BASELINE configs[1] (cosmics, 70x70 pixels, 30 cm drift, noise on): all segment stages, and the
    currents of a sample of pixels (the busiest ones plus a random draw) against the oracle."""
    wl = W.make_config(1)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response=mode)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm, max_pixels=48)
    sim.close()


@pytest.mark.parametrize("mode", MODES)
def test_zero_drift_and_edges(lartpc, mode):
    """Degenerate cases: segments at the anode (sigma = 0, indicator weights), at the plane edge (charge bins
    outside the plane act on in-plane pixels), outside every TPC, zero length and zero energy."""
    p = W.default_params(n_readout_ticks=900)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, 10.0, 16, 16, 0)]
    pitch = p["pixel_pitch_cm"]
    rng = np.random.Generator(np.random.PCG64(3))
    parts = [
        W.line_segments([3.3 * pitch, 4.2 * pitch, 0.0], [6.1 * pitch, 5.9 * pitch, 0.0], 0.1, 0.5, W._mip(2.1)),  # anode
        W.line_segments([0.05 * pitch, 7.0 * pitch, 4.0], [2.0 * pitch, 7.7 * pitch, 4.3], 0.1, 0.0, W._mip(2.1)),  # left edge
        W.line_segments([14.0 * pitch, 15.95 * pitch, 2.0], [15.9 * pitch, 15.6 * pitch, 2.5], 0.1, 0.0, W._mip(2.1)),  # corner
        W.line_segments([30.0, 1.0, 1.0], [30.5, 1.0, 1.0], 0.1, 0.0, W._mip(2.1)),                                  # outside
    ]
    seg = W._concat(parts)
    for k in seg:
        seg[k] = np.concatenate([seg[k], seg[k][:2]])
    seg["xe"][-1] = seg["xs"][-1]; seg["ye"][-1] = seg["ys"][-1]; seg["ze"][-1] = seg["zs"][-1]    # zero length
    seg["dE"][-2] = 0.0                                                                               # zero energy
    wl = W.Workload("edges", 5, p, tpcs, seg, W.pad_response_lut(p))
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response=mode)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm)
    _check_hits(res, wl, dr, pm, wl.seed)
    sim.close()


def test_empty_input(lartpc):
    wl = W.make_config(0)
    wl = wl.subset(np.zeros(0, dtype=np.int64))
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, wl)
    assert res["n_active"] == 0 and int(res["hits"]["counters"][0]) == 0 and res["info"].n_tiles == 0
    seg = sim.upload_segments(wl.segments)
    hits, st = sim.run_spill(seg, 1, hit_capacity=16)
    assert st.n_hits == 0
    sim.close()


def test_short_drift_all_node_rules(lartpc):
    """The tensor-core splat replaces a segment's N midpoints by an n-node rule chosen from its extent over the
    diffusion sigma (n = 8 .. 32, or its own midpoints when the segment is sharp or short).  Tracks along x, along the
    drift direction and oblique, at 0.2 .. 8 cm of drift, with 1 mm, 0.5 mm and 0.25 mm segments, walk through every
    rule and the fall-back; every pixel is compared with the oracle (which always sums the N midpoints)."""
    p = W.default_params(n_readout_ticks=1400)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, 12.0, 24, 24, 0)]
    pitch = p["pixel_pitch_cm"]
    parts = []
    for k, (z, step) in enumerate([(0.2, 0.1), (0.5, 0.1), (1.0, 0.1), (2.0, 0.1), (4.0, 0.1), (8.0, 0.1),
                                   (0.5, 0.05), (2.0, 0.05), (8.0, 0.025)]):
        y = (2.2 + 2.1 * k) * pitch
        parts.append(W.line_segments([3.1 * pitch, y, z], [6.3 * pitch, y + 0.013, z], step, 0.0, W._mip(2.1)))        # along x
        parts.append(W.line_segments([9.4 * pitch, y, z], [9.4 * pitch + 0.01, y + 0.02, z + 0.6], step, 0.0, W._mip(2.1)))  # along the drift
        parts.append(W.line_segments([13.2 * pitch, y, z], [15.9 * pitch, y + 0.5 * pitch, z + 0.35], step, 0.0, W._mip(6.0)))  # oblique
    # long segments (10 mm at 8 cm, 5 mm at 1 cm of drift): beyond the largest rule, they keep their own midpoints
    parts.append(W.line_segments([2.2 * pitch, 21.3 * pitch, 8.0], [11.0 * pitch, 22.1 * pitch, 8.9], 1.0, 0.0, W._mip(2.1)))
    parts.append(W.line_segments([14.2 * pitch, 21.6 * pitch, 1.0], [17.5 * pitch, 22.4 * pitch, 1.3], 0.5, 0.0, W._mip(2.1)))
    seg = W._concat(parts)
    wl = W.Workload("short-drift", 6, p, tpcs, seg, W.pad_response_lut(p))
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm)
    _check_hits(res, wl, dr, pm, wl.seed)
    sim.close()


@pytest.mark.parametrize("window,lut_ticks,mode", [(9, 200, "tensor"), (9, 200, "ffma"), (5, 500, "ffma"), (5, 120, "tensor"),
                                                   (5, 500, "tensor"), (5, 1000, "tensor"), (9, 300, "tensor")])
def test_config4_axes_small(lartpc, window, lut_ticks, mode):
    """BASELINE configs[4] sweep axes at a size the oracle finishes in seconds: 9x9 response window and LUT lengths
    other than 200 ticks (K > 241: the tensor-core path cuts the LUT into pieces of 200 ticks, each a row of its own that S5
    adds; the FFMA2 kernel takes any length as it is)."""
    p = W.default_params(window_pixels=window, lut_ticks=lut_ticks, n_readout_ticks=700 + lut_ticks)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, 20.0, 20, 20, 0)]
    pitch = p["pixel_pitch_cm"]
    parts = [W.line_segments([2.3 * pitch, 3.1 * pitch, 6.0], [9.7 * pitch, 12.4 * pitch, 7.5], 0.1, 0.0, W._mip(2.1)),
             W.line_segments([15.2 * pitch, 1.1 * pitch, 1.0], [18.9 * pitch, 3.0 * pitch, 1.2], 0.05, 0.3, W._mip(8.0))]
    wl = W.Workload("c4-small", 4, p, tpcs, W._concat(parts), W.pad_response_lut(p))
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response=mode)
    assert sim.response_mode == mode
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_currents(res, wl, dr, pm, max_pixels=40)
    sim.close()


def _sampled_hits_check(lartpc_mod, wl, res, dr, pm, per_tpc, seed, only_tpcs=None):
    """Currents and hits of a sample of pixels per TPC (the busiest ones plus a random draw) against O4-O6."""
    nt = wl.params["n_readout_ticks"]
    gpu_ids = res["waveforms"]["pixel_id"][:res["n_active"]]
    disabled = set() if wl.disabled_pixels is None else set(int(x) for x in wl.disabled_pixels)
    dense_q = res["hits"]["q_pixel"][:res["n_active"]]
    rng = np.random.Generator(np.random.PCG64(seed))
    h = res["hits"]
    n = int(h["counters"][0])
    ghits = {}
    for p_, t_, a_ in zip(h["hit_pixel"][:n].tolist(), h["hit_tick"][:n].tolist(), h["hit_adc"][:n].tolist()):
        ghits.setdefault(p_, []).append((t_, a_))
    assert not any(p_ in disabled for p_ in ghits), "a disabled pixel produced a hit"
    n_o = n_same = 0
    worst_q = 0.0
    wf = res["waveforms"]
    for ti, t in enumerate(wl.tpcs):
        if only_tpcs is not None and ti not in only_tpcs:
            continue
        sel = np.nonzero((gpu_ids >= t["first_pixel_id"]) & (gpu_ids < t["first_pixel_id"] + t["nx"] * t["ny"]))[0]
        sel = np.array([i for i in sel if int(gpu_ids[i]) not in disabled], dtype=np.int64)
        if len(sel) == 0:
            continue
        if len(sel) > per_tpc:
            top = sel[np.argsort(np.abs(dense_q[sel]))[-per_tpc // 2:]]
            rest = rng.choice(sel, size=per_tpc // 2, replace=False)
            sel = np.unique(np.concatenate([top, rest]))
        rel = gpu_ids[sel] - t["first_pixel_id"]
        waves, qp = oracle.pixel_currents(wl.params, wl.tpcs, wl.lut, dr, pm, ti, rel % t["nx"], rel // t["nx"])
        gq = np.zeros(len(sel))
        for k, i in enumerate(sel):
            o, f, l = int(wf["offset"][i]), int(wf["first_tick"][i]), int(wf["length"][i])
            g = np.zeros(nt)
            g[f:f + l] = wf["samples"][o:o + l]
            gq[k] = g.sum()
            peak = np.abs(waves[k]).max()
            assert np.all(np.abs(g - waves[k]) <= 1e-4 * peak + 0.02)
        tol = np.maximum(1e-4 * np.abs(qp), 1.0)
        assert np.all(np.abs(gq - qp) <= tol), (np.abs(gq - qp) / tol).max()
        worst_q = max(worst_q, float((np.abs(gq - qp) / tol).max()))
        hp, ht, ha, _ = oracle.electronics(wl.params, seed, gpu_ids[sel].astype(np.int32), waves)
        for p_, t_, a_ in zip(hp.tolist(), ht.tolist(), ha.tolist()):
            n_o += 1
            got = ghits.get(p_, [])
            if (t_, a_) in got:
                n_same += 1
            else:
                assert any(abs(t2 - t_) <= 1 and abs(a2 - a_) <= 1 for t2, a2 in got), (p_, t_, a_, got)
        ohits = {}
        for p_, t_ in zip(hp.tolist(), ht.tolist()):
            ohits[p_] = ohits.get(p_, 0) + 1
        for i in sel:
            assert len(ghits.get(int(gpu_ids[i]), [])) == ohits.get(int(gpu_ids[i]), 0)
    assert n_o > 0 and n_same >= 0.999 * n_o, (n_same, n_o)
    print("sampled pixels: worst |dQ| / tol = %.3f, %d / %d oracle hits identical" % (worst_q, n_same, n_o))


def test_config2_sampled_full_chain(lartpc):
    """BASELINE configs[2] at full size (1e5 segments, 8 TPCs, Birks, noise on, 7.8 % of the pixels disabled): every
    segment-stage output, the currents and hits of a sample of pixels per TPC against the oracle, and the hit list of
    lartpc_run_spill (TPC batches) against the staged calls."""
    wl = W.make_config(2)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    sim.set_disabled_pixels(wl.disabled_pixels)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _sampled_hits_check(lartpc, wl, res, dr, pm, per_tpc=12, seed=wl.seed)
    seg = sim.upload_segments(wl.segments)
    hits, st = sim.run_spill(seg, wl.seed, hit_capacity=1 << 20)
    n = int(res["hits"]["counters"][0])
    assert st.n_hits == n and st.n_hits_dropped == 0
    for a, k in zip(lartpc.hits_to_numpy(hits), ("hit_pixel", "hit_tick", "hit_adc")):
        assert np.array_equal(a, res["hits"][k][:n])
    sim.close()


def test_config3_full_spill(lartpc):
    """BASELINE configs[3] at full size, in the configuration bench.py times (lartpc_run_spill over 70 TPCs in batches).
    The oracle cannot do 5e6 segments, so: (a) the two busiest TPCs are simulated alone through the staged calls, at
    their full density, and a sample of their pixels is held to the oracle (currents and hits); (b) the full spill's hits
    on those two TPCs must be the staged ones bit for bit (batching, tile sorting and the slot map change no result);
    (c) properties of the whole list: sorted by (pixel, tick), nothing dropped, ADC within 8 bits, ticks inside the window."""
    wl = W.make_config(3)
    _, ne = oracle.quench(wl.params, wl.segments)
    tpc_of = oracle.drift(wl.params, wl.tpcs, wl.segments, ne)["tpc"]
    counts = np.bincount(tpc_of[tpc_of >= 0], minlength=len(wl.tpcs))
    busy = [int(x) for x in np.argsort(counts)[-2:]]
    sub = wl.subset(np.nonzero(np.isin(tpc_of, busy))[0])
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, sub)
    dr, pm = _check_segment_stages(res, sub)
    _sampled_hits_check(lartpc, sub, res, dr, pm, per_tpc=10, seed=wl.seed, only_tpcs=busy)
    n_sub = int(res["hits"]["counters"][0])
    sub_hits = [res["hits"][k][:n_sub].copy() for k in ("hit_pixel", "hit_tick", "hit_adc")]
    del res
    import torch
    torch.cuda.empty_cache()
    seg = sim.upload_segments(wl.segments)
    hits, st = sim.run_spill(seg, wl.seed, hit_capacity=int(8 * wl.n_segments))
    assert st.n_hits > 0 and st.n_hits_dropped == 0 and st.n_batches >= 1
    # pixels with more than max_hits_per_pixel hits are counted, never silent (D18): a handful in the shower cores
    assert st.n_pixels_overflow <= 1e-4 * st.n_active_pixels and st.n_hits_total - st.n_hits >= st.n_pixels_overflow
    hp, ht, ha = lartpc.hits_to_numpy(hits)
    key = hp.astype(np.int64) * (1 << 20) + ht
    assert np.all(np.diff(key) > 0)
    assert ha.min() >= 0 and ha.max() <= 255 and ht.min() >= 0 and ht.max() < wl.params["n_readout_ticks"]
    in_busy = np.zeros(len(hp), dtype=bool)
    for ti in busy:
        t = wl.tpcs[ti]
        in_busy |= (hp >= t["first_pixel_id"]) & (hp < t["first_pixel_id"] + t["nx"] * t["ny"])
    assert in_busy.sum() == n_sub
    assert np.array_equal(hp[in_busy], sub_hits[0]) and np.array_equal(ht[in_busy], sub_hits[1]) and np.array_equal(ha[in_busy], sub_hits[2])
    # (d) the 16-bit packed output of the whole spill (70 x 70 readout tiles, partial tiles at the plane edges)
    packed, offs = sim.pack_hits(hits, st.n_hits, 70)
    want_p, want_o = _pack_reference(wl, hp, ht, ha, 70)
    assert np.array_equal(offs.cpu().numpy(), want_o) and np.array_equal(packed.cpu().numpy().view(np.uint16), want_p)
    print("config 3: %d segments, %d tiles, %d hits; TPCs %s alone: %d hits, identical inside the full spill"
          % (wl.n_segments, st.n_tiles, st.n_hits, busy, n_sub))
    sim.close()


@pytest.mark.parametrize("variant", ["disc_noise", "periodic_reset", "low_threshold"])
def test_electronics_variants(lartpc, variant):
    """SURVEY 8(f) NEXT-4 options of S6: discriminator noise 650 e- (drawn every tick, so the
    per-tick kernel runs instead of the warp-scan one), the periodic reset, and the low-threshold regime."""
    over = dict(noise_reset_e=900.0, noise_uncorr_e=500.0)
    if variant == "disc_noise":
        over.update(noise_disc_e=650.0)
    elif variant == "periodic_reset":
        over.update(periodic_reset_ticks=97)
    else:
        over.update(threshold_e=3000.0, min_spacing_ticks=11)
    wl = W.make_config(0, seed=11)
    wl.params.update(over)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    _check_hits(res, wl, dr, pm, wl.seed)
    sim.close()


@pytest.mark.parametrize("m,seed", [(1, 5), (3, 0xABCDEF0123)])
def test_random_perturbations_same_draws(lartpc, m, seed):
    """SURVEY 8(f) NEXT-1, eq. (3.9) as printed: M random perturbations per sample point, nearest-bin look-up.
    Both sides key the normals by (seed; segment, mu, nu) (reading D25), so the comparison is draw for draw: the waveforms
    and charges of every active pixel, and the hits, against the oracle's random estimator."""
    wl = W.make_config(0, seed=21)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    sim.set_random_perturbations(m, seed)
    res = run_staged(sim, wl)
    dr, pm = _check_segment_stages(res, wl)
    nt = wl.params["n_readout_ticks"]
    dense = dense_waves(res, nt)
    gpu_ids = res["waveforms"]["pixel_id"][:res["n_active"]]
    t = wl.tpcs[0]
    rel = gpu_ids - t["first_pixel_id"]
    waves, qp = oracle.pixel_currents_random(wl.params, wl.tpcs, wl.lut, dr, pm, 0, rel % t["nx"], rel // t["nx"], m, seed)
    assert qp.sum() > 0
    gq = dense.sum(axis=1)
    tol = np.maximum(1e-4 * np.abs(qp), 1.0)
    assert np.all(np.abs(gq - qp) <= tol), (np.abs(gq - qp) / tol).max()
    peak = np.abs(waves).max(axis=1, keepdims=True)
    assert np.all(np.abs(dense - waves) <= 1e-4 * peak + 0.02)
    # it is a different estimate from the expectation form, not the same numbers
    _, q_exp = oracle.pixel_currents(wl.params, wl.tpcs, wl.lut, dr, pm, 0, rel % t["nx"], rel // t["nx"])
    assert np.abs(qp - q_exp).max() > 10.0 and qp.sum() == pytest.approx(q_exp.sum(), rel=1e-5)
    hp, ht, ha, _ = oracle.electronics(wl.params, wl.seed, gpu_ids.astype(np.int32), waves)
    h = res["hits"]
    n = int(h["counters"][0])
    frac, near, ng, no = compare_hits((h["hit_pixel"][:n], h["hit_tick"][:n], h["hit_adc"][:n]), (hp, ht, ha))
    assert no > 0 and frac >= 0.999 and near and ng == no
    # back to the default
    sim.set_random_perturbations(0)
    res0 = run_staged(sim, wl)
    assert np.allclose(dense_waves(res0, nt).sum(axis=1), q_exp, rtol=1e-4, atol=1.0)
    sim.close()


def test_random_perturbations_need_the_tensor_path(lartpc):
    wl = W.make_config(0)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response="ffma")
    with pytest.raises(lartpc.LartpcError):
        sim.set_random_perturbations(2, 1)
    sim.close()


def _pack_reference(wl, hp, ht, ha, tile_pixels):
    """The packed layout written out with numpy from its definition (include/lartpc.h, lartpc_pack_hits)."""
    tile_of, in_tile = np.zeros(len(hp), dtype=np.int64), np.zeros(len(hp), dtype=np.int64)
    base = 0
    for t in wl.tpcs:
        ntx, nty = -(-t["nx"] // tile_pixels), -(-t["ny"] // tile_pixels)
        m = (hp >= t["first_pixel_id"]) & (hp < t["first_pixel_id"] + t["nx"] * t["ny"])
        rel = hp[m].astype(np.int64) - t["first_pixel_id"]
        iy, ix = rel // t["nx"], rel % t["nx"]
        tile_of[m] = base + (iy // tile_pixels) * ntx + ix // tile_pixels
        in_tile[m] = (iy % tile_pixels) * tile_pixels + ix % tile_pixels
        base += ntx * nty
    order = np.lexsort((ht, in_tile, tile_of))
    packed = np.stack([in_tile[order], ht[order], ha[order] & 0x0fff], axis=1).astype(np.uint16)
    offs = np.concatenate([[0], np.cumsum(np.bincount(tile_of, minlength=base))]).astype(np.int64)
    return packed, offs


@pytest.mark.parametrize("tile_pixels", [70, 32])
def test_packed_hit_output(lartpc, tile_pixels):
    """BASELINE configs[3] "16-bit packed hit output" (D18) on the configs[2] spill: three uint16 per hit grouped by
    readout tile with an offset table, bit-exact against the layout's definition; partial tiles at the plane edges."""
    wl = W.make_config(2)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    seg = sim.upload_segments(wl.segments)
    hits, st = sim.run_spill(seg, wl.seed, hit_capacity=1 << 20)
    packed, offs = sim.pack_hits(hits, st.n_hits, tile_pixels)
    hp, ht, ha = lartpc.hits_to_numpy(hits, st.n_hits)
    want_p, want_o = _pack_reference(wl, hp, ht, ha, tile_pixels)
    assert st.n_hits > 1000
    assert np.array_equal(offs.cpu().numpy(), want_o)
    assert np.array_equal(packed.cpu().numpy().view(np.uint16), want_p)
    # empty list
    packed0, offs0 = sim.pack_hits(hits, 0, tile_pixels)
    assert packed0.shape[0] == 0 and np.all(offs0.cpu().numpy() == 0)
    sim.close()
