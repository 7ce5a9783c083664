"""GPU parity of the light simulation (eqs. 4.1-4.6) against oracle O8-O12, stage by stage through the
C-ABI, on seeded workloads with the synthetic light LUT of workloads.light_setup.

Tolerances: voxel and tick indices bit-exact (float64 index path on both sides); N_gamma, N_pe 2e-6
relative (float32 storage of n_e and of the result); the time profile and the two convolutions 1e-5 of the waveform's peak
(float32 sums of up to a few thousand terms in a fixed order against float64); the counting statistics are compared on the
SAME float32 means: Poisson counts identical, normal samples 2e-6 relative + 1e-4 absolute; the chained waveform is held to the
oracle run on the GPU's own observed photoelectrons (the chain's one discrete step is checked separately)."""
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


def _gpu_stages(lartpc, wl, ls, seed):
    import torch
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut)
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    light = lartpc.LightSim(ls.params, ls.eff, ls.gain, ls.vis, ls.tprof, ls.resp, ls.noise_amp, ls.noise_k)
    a = light.npe(seg, ne)
    ipe = light.profile(a)
    isc = light.scintillation(ipe)
    nobs = light.fluctuate(isc, seed)
    v = light.electronics(nobs, seed)
    v_run = light.run(seg, ne, seed)
    v_again = light.run(seg, ne, seed)
    torch.cuda.synchronize()
    assert torch.equal(v_run, v_again)                              # fixed summation order: bit-identical from run to run
    out = dict(vox=a["vox"].cpu().numpy(), k0=a["k0"].cpu().numpy(), n_gamma=a["n_gamma"].cpu().numpy(),
               npe=a["npe"].cpu().numpy(), ipe=ipe.cpu().numpy(), isc=isc.cpu().numpy(), nobs=nobs.cpu().numpy(),
               v=v.cpu().numpy(), v_run=v_run.cpu().numpy(), n_e=ne.cpu().numpy())
    light.close()
    sim.close()
    return out


def _check(wl, ls, g, seed):
    lp = ls.params
    _, ne = oracle.quench(wl.params, wl.segments)
    o = oracle.light_npe(lp, wl.segments, ne, ls.eff, ls.vis)
    assert np.array_equal(g["vox"], o["vox"]) and np.array_equal(g["k0"], o["k0"])
    assert np.allclose(g["n_gamma"], o["n_gamma"], rtol=2e-6, atol=1e-3)
    assert np.allclose(g["npe"], o["npe"], rtol=4e-6, atol=1e-9 + 2e-6 * np.abs(o["npe"]).max())
    # eq. (4.3)
    ipe = oracle.light_profile(lp, o["vox"], o["k0"], o["npe"], ls.tprof)
    assert ipe.max() > 0
    assert np.all(np.abs(g["ipe"] - ipe) <= 1e-5 * ipe.max(axis=1, keepdims=True) + 1e-12)
    # eq. (4.5)
    w = oracle.light_scint_weights(lp)
    isc = oracle.light_convolve(ipe, w)
    assert np.all(np.abs(g["isc"] - isc) <= 1e-5 * isc.max(axis=1, keepdims=True) + 1e-12)
    # counting statistics on the GPU's own float32 means: same uniforms, same float64 decisions
    nobs = oracle.light_fluctuate(lp, seed, g["isc"].astype(np.float64))
    pois = (g["isc"] > 0) & (g["isc"] < lp["normal_above"])
    norm = g["isc"] >= lp["normal_above"]
    assert np.array_equal(g["nobs"][pois], nobs[pois].astype(np.float32))
    assert np.all(g["nobs"][g["isc"] <= 0] == 0)
    if norm.any():
        assert np.allclose(g["nobs"][norm], nobs[norm], rtol=2e-6, atol=1e-4)
    # and how often the two chains agree end to end (means differ by ~1e-6 relative: a count flips when u sits on a CDF step)
    nobs_chain = oracle.light_fluctuate(lp, seed, isc)
    both = pois & (isc > 0) & (isc < lp["normal_above"])
    mismatch = float((g["nobs"][both] != nobs_chain[both]).mean()) if both.any() else 0.0
    assert mismatch <= 1e-4, mismatch
    # eq. (4.6) on the GPU's observed photoelectrons
    v = oracle.light_convolve(g["nobs"].astype(np.float64), ls.resp.astype(np.float64), ls.gain)
    if int(lp["n_noise"]) > 0:
        v = v + oracle.light_noise(lp, seed, ls.noise_amp, ls.noise_k)
    scale = np.abs(v).max(axis=1, keepdims=True) + 1e-9
    assert np.all(np.abs(g["v"] - v) <= 2e-5 * scale)
    assert np.array_equal(g["v_run"], g["v"])                       # lartpc_light_run == the staged calls, bit for bit
    return dict(pe=float(o["npe"].sum()), poisson=int(pois.sum()), normal=int(norm.sum()), mismatch=mismatch)


@pytest.mark.parametrize("cfg,n_det,noise,eff_scale", [(0, 6, False, 1.0), (0, 6, True, 600.0), (1, 12, True, 1.0)])
def test_light_chain_small(lartpc, cfg, n_det, noise, eff_scale):
    """configs[0] (one track; with the efficiencies scaled up the normal branch of P:L782 is reached) and configs[1]
    (20 muons): every stage against the oracle."""
    wl = W.make_config(cfg)
    ls = W.light_setup(wl, n_det=n_det, noise=noise)
    ls.eff = (ls.eff * eff_scale).astype(np.float32)
    g = _gpu_stages(lartpc, wl, ls, wl.seed)
    r = _check(wl, ls, g, wl.seed)
    assert r["poisson"] > 100 and (eff_scale == 1.0 or r["normal"] > 50)
    print("light configs[%d]: %.0f p.e., %d Poisson / %d normal samples, chain mismatch %.1e" % (cfg, r["pe"], r["poisson"], r["normal"], r["mismatch"]))


def test_light_edges(lartpc):
    """Segments outside the voxel grid (no light), before tick 0 (their light partly or wholly before the waveform), at its
    end (light running past the last tick), zero energy; lut_m = 3, a LUT of 5 bins; empty input."""
    wl = W.make_config(0)
    seg = {k: v.copy() for k, v in wl.segments.items()}
    n = len(seg["xs"])
    seg["ts"][:10] = seg["te"][:10] = -0.40          # before t_start = -0.32: k0 < 0
    seg["ts"][10:20] = seg["te"][10:20] = -0.33      # k0 = -1
    seg["dE"][20:25] = 0.0
    seg["xs"][25:30] += 500.0
    seg["xe"][25:30] += 500.0                        # outside the grid
    ls = W.light_setup(wl, n_det=5, lut_m=3, n_lut_t=5, noise=False)
    t_end = ls.params["t_start_us"] + ls.params["n_ticks"] * ls.params["tick_us"]
    seg["ts"][30:40] = seg["te"][30:40] = t_end - 0.05   # light runs past the last tick
    seg["ts"][40:45] = seg["te"][40:45] = t_end + 1.0    # after the waveform
    import dataclasses
    wl2 = dataclasses.replace(wl, segments=seg)
    g = _gpu_stages(lartpc, wl2, ls, 3)
    r = _check(wl2, ls, g, 3)
    assert (g["vox"] < 0).sum() == 5 and (g["k0"] < 0).sum() == 20
    # empty input
    empty = wl.subset(np.zeros(0, dtype=np.int64))
    g0 = _gpu_stages(lartpc, empty, ls, 3)
    assert not g0["ipe"].any() and not g0["v"].any()
    assert n == 100 and r["pe"] > 0


def test_light_config2(lartpc):
    """BASELINE configs[2] (1e5 segments, 8 TPCs): 16 sensors, the whole chain against the oracle."""
    wl = W.make_config(2)
    ls = W.light_setup(wl, n_det=16, noise=True)
    ls.eff = (ls.eff * 25.0).astype(np.float32)                     # bright enough for both branches of P:L782
    g = _gpu_stages(lartpc, wl, ls, wl.seed)
    r = _check(wl, ls, g, wl.seed)
    assert r["normal"] > 300 and r["poisson"] > 1000
    print("light configs[2]: %.3g p.e., %d Poisson / %d normal samples, chain mismatch %.1e" % (r["pe"], r["poisson"], r["normal"], r["mismatch"]))
