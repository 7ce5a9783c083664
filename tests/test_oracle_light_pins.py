"""Pins of the light-simulation oracle (O8-O12 of oracle/lartpc_oracle.c, readings
D28-D33): every function is held to something other than itself -- closed forms, hand-placed inputs, conservation,
numpy / scipy library routines, the test's own Philox."""
import math

import numpy as np
import pytest

import oracle
from paper_2212_09807_b200 import workloads as W
from test_oracle_pins import _philox_py

LGHT = 0x4C474854


def _lp(**over):
    return W.default_light_params(**over)


def _seg(rows):
    """rows: (xs, ys, zs, ts, xe, ye, ze, te, dE)"""
    a = np.asarray(rows, dtype=np.float32)
    return {k: np.ascontiguousarray(a[:, i]) for i, k in enumerate(W.SEG_FIELDS)}


def test_light_photon_yield_and_voxels_by_hand():
    """Eqs. (4.1)(4.2): a 1 cm MIP piece (2.1 MeV) with the modified Box recombination of eq. (3.2) worked here:
    xi = 0.212 x 2.1 / (0.5 x 1.38), R = ln(0.93 + xi) / xi = 0.7042; N_gamma = dE / W_ph - R dE / W_ion =
    107 692 - 62 666 = 45 026 photons; N_pe = eps_i V_i[voxel] N_gamma with the voxel of the midpoint (D28)."""
    p = W.default_params()
    lp = _lp(nvx=3, nvy=2, nvz=2, vox_size_cm=4.0, vox_x0=-2.0, vox_y0=0.0, vox_z0=10.0, n_det=2, t_start_us=-0.32, tick_us=0.016)
    seg = _seg([(1.0, 1.0, 11.0, 0.10, 2.0, 1.0, 11.0, 0.12, 2.1),          # midpoint (1.5, 1, 11) -> voxel (0, 0, 0)
                (9.0, 5.0, 15.0, 0.0, 9.0, 6.0, 15.0, 0.0, 2.1),            # midpoint (9, 5.5, 15) -> voxel (2, 1, 1) = 11
                (11.0, 1.0, 11.0, 0.0, 12.0, 1.0, 11.0, 0.0, 2.1),          # x = 11.5: outside the 12 cm grid that starts at -2
                (1.0, 1.0, 11.0, 0.0, 2.0, 1.0, 11.0, 0.0, 0.0)])           # no energy
    _, ne = oracle.quench(p, seg)
    xi = 0.212 * 2.1 / (0.5 * 1.38)
    R = math.log(0.93 + xi) / xi
    assert R == pytest.approx(0.7042, abs=2e-4) and ne[0] == pytest.approx(R * 2.1 / 23.6e-6, rel=1e-6)
    n_gamma = 2.1 / 19.5e-6 - R * 2.1 / 23.6e-6
    assert n_gamma == pytest.approx(45026, abs=30)
    eff = np.array([0.004, 0.25], dtype=np.float32)
    vis = np.zeros((2, 2, 2, 3), dtype=np.float32)
    vis[0, 0, 0, 0], vis[1, 0, 0, 0], vis[0, 1, 1, 2], vis[1, 1, 1, 2] = 0.5, 0.125, 0.03125, 1.0
    a = oracle.light_npe(lp, seg, ne, eff, vis)
    assert a["vox"].tolist() == [0, 11, -1, 0]
    assert a["k0"].tolist() == [math.floor((0.11 + 0.32) / 0.016), 20, 20, 20]
    assert np.allclose(a["n_gamma"][:2], n_gamma, rtol=1e-6) and a["n_gamma"][3] == 0.0
    want = np.array([[np.float32(0.004) * 0.5 * n_gamma, np.float32(0.004) * 0.03125 * n_gamma, 0.0, 0.0],
                     [0.25 * 0.125 * n_gamma, 0.25 * 1.0 * n_gamma, 0.0, 0.0]])
    assert np.allclose(a["npe"], want, rtol=1e-6)
    # more charge means less light: the anticorrelation of eq. (4.1)
    assert a["n_gamma"][0] + ne[0] == pytest.approx(float(seg["dE"][0]) / 19.5e-6, rel=1e-12)


def test_light_profile_by_hand_and_conservation():
    """Eq. (4.3) as read in D29: a segment with k0 = 5 and N_pe = 8 under f = (0.5, 0.25, 0.25), lut_m = 2, puts
    2, 2, 1, 1, 1, 1 photoelectrons into ticks 5 .. 10; light that would land outside the waveform is dropped; the sum over
    ticks is the sum of N_pe for everything inside."""
    lp = _lp(n_det=2, n_ticks=16, lut_m=2, n_lut_t=3, nvx=2, nvy=1, nvz=1)
    tprof = np.zeros((2, 2, 3), dtype=np.float32)
    tprof[0, 0] = (0.5, 0.25, 0.25)
    tprof[0, 1] = (0.0, 1.0, 0.0)
    tprof[1, :] = (0.25, 0.25, 0.5)
    vox = np.array([0, 1, -1, 0], dtype=np.int32)
    k0 = np.array([5, 0, 3, 13], dtype=np.int32)
    npe = np.array([[8.0, 3.0, 100.0, 4.0], [0.0, 2.0, 100.0, 0.0]])
    ipe = oracle.light_profile(lp, vox, k0, npe, tprof)
    want0 = np.zeros(16)
    want0[5:11] = (2, 2, 1, 1, 1, 1)
    want0[2:4] += 1.5                                   # segment 1: all of its 3 p.e. in LUT bin 1 = ticks 2, 3
    want0[13:15] += 1.0                                 # segment 3: bin 0 in ticks 13, 14; bins 1 and 2 run past tick 15
    want0[15] += 0.5
    assert np.allclose(ipe[0], want0, rtol=0, atol=1e-12)
    want1 = np.zeros(16)
    want1[0:4] = 0.25
    want1[4:6] = 0.5
    assert np.allclose(ipe[1], want1, atol=1e-12)
    assert ipe[1].sum() == pytest.approx(2.0) and ipe[0].sum() == pytest.approx(8 + 3 + 4 * (0.5 + 0.125))


def test_light_scintillation_weights_closed_forms():
    """Eq. (4.4) integrated over a tick (D30): w[0] = f_p (1 - e^{-dt/tau_p}) + (1 - f_p)(1 - e^{-dt/tau_s}); the weights
    telescope to 1 - f_p e^{-(S+1) dt/tau_p} - (1 - f_p) e^{-(S+1) dt/tau_s} > 0.99 with S = floor(5 tau_s / dt) (P:L769
    "> 99 % of the total light"); for dt << tau_p they agree with f_scint(s dt) dt as eq. (4.5) prints it."""
    for dt in (0.016, 0.001):
        lp = _lp(tick_us=dt)
        w = oracle.light_scint_weights(lp)
        S = int(math.floor(5.0 * 1.6 / dt))
        assert len(w) == S + 1
        assert w[0] == pytest.approx(0.3 * (1 - math.exp(-dt / 0.007)) + 0.7 * (1 - math.exp(-dt / 1.6)), rel=1e-12)
        total = 1 - 0.3 * math.exp(-(S + 1) * dt / 0.007) - 0.7 * math.exp(-(S + 1) * dt / 1.6)
        assert w.sum() == pytest.approx(total, rel=1e-12) and 0.99 < w.sum() < 1.0
        assert np.all(np.diff(w) < 0)
    lp = _lp(tick_us=1e-4)
    w = oracle.light_scint_weights(lp)
    s = np.arange(len(w)) * 1e-4
    printed = (0.3 / 0.007 * np.exp(-s / 0.007) + 0.7 / 1.6 * np.exp(-s / 1.6)) * 1e-4
    assert np.allclose(w, printed, rtol=8e-3)               # first order in dt / tau_p = 1.4e-2


def test_light_convolution_against_numpy():
    """Eq. (4.5) / the sum of eq. (4.6): the truncated causal convolution is numpy's full convolution cut to the waveform;
    an impulse returns the weights, scaled by G_i."""
    rng = np.random.Generator(np.random.PCG64(11))
    x = rng.uniform(0, 5, size=(3, 200))
    w = rng.uniform(0, 1, size=37)
    g = np.array([1.0, 2.5, 0.5], dtype=np.float32)
    got = oracle.light_convolve(x, w, g)
    for i in range(3):
        assert np.allclose(got[i], g[i] * np.convolve(x[i], w)[:200], rtol=1e-12, atol=1e-12)
    imp = np.zeros((1, 64))
    imp[0, 10] = 3.0
    out = oracle.light_convolve(imp, w)
    assert np.allclose(out[0, 10:47], 3.0 * w) and not out[0, :10].any() and not out[0, 47:].any()
    # a constant input under the scintillation weights settles at (sum of weights) x input
    lp = _lp()
    ws = oracle.light_scint_weights(lp)
    y = oracle.light_convolve(np.full((1, 700), 2.0), ws)
    assert y[0, 650] == pytest.approx(2.0 * ws.sum(), rel=1e-12)


def test_light_poisson_is_the_inverse_cdf_and_normal_by_hand():
    """P:L782.  Below 30 expected photoelectrons the inverse-transform sample is the smallest k with CDF(k) >= u:
    scipy.stats.poisson.ppf at the uniform the test derives from its own Philox; at and above 30 the sample is
    lambda + sqrt(lambda) z with the Box-Muller normal of (u0, u1); lambda <= 0 gives nothing."""
    from scipy.stats import poisson
    lp = _lp(n_det=4, n_ticks=64)
    seed = 0x1234567890ABCDEF
    rng = np.random.Generator(np.random.PCG64(3))
    lam = rng.uniform(0.0, 29.9, size=(4, 64))
    lam[0, :8] = (0.0, -1.0, 1e-6, 0.01, 29.99, 30.0, 31.0, 5000.0)
    got = oracle.light_fluctuate(lp, seed, lam)
    n_pois = 0
    for i in range(4):
        for t in range(64):
            x = _philox_py((i, t, 0, LGHT), (seed & 0xFFFFFFFF, seed >> 32))
            u0, u1 = (x[0] + 0.5) / 4294967296.0, (x[1] + 0.5) / 4294967296.0
            l = lam[i, t]
            if l <= 0:
                assert got[i, t] == 0.0
            elif l < 30.0:
                assert got[i, t] == poisson.ppf(u0, l), (i, t, l, u0)
                n_pois += 1
            else:
                z = math.sqrt(-2 * math.log(u0)) * math.cos(2 * math.pi * u1)
                assert got[i, t] == pytest.approx(l + math.sqrt(l) * z, rel=1e-12)
    assert n_pois > 200
    # moments over many keys: mean and variance of a Poisson(4.5)
    lp2 = _lp(n_det=8, n_ticks=4096)
    s = oracle.light_fluctuate(lp2, 99, np.full((8, 4096), 4.5))
    assert s.mean() == pytest.approx(4.5, abs=0.05) and s.var() == pytest.approx(4.5, abs=0.15)
    s = oracle.light_fluctuate(lp2, 99, np.full((8, 4096), 400.0))
    assert s.mean() == pytest.approx(400.0, abs=0.5) and s.std() == pytest.approx(20.0, abs=0.4)


def test_light_noise_by_hand():
    """Reading D33: n_i[t] = sum_f A_f cos(2 pi k_f t / n_ticks + phi_if), phi_if = 2 pi u_0 of Philox(counter (i, f, 1,
    'LGHT')); its mean square is sum A_f^2 / 2 for integer k_f."""
    lp = _lp(n_det=2, n_ticks=256, n_noise=2)
    amp, kf = np.array([3.0, 0.5], dtype=np.float32), np.array([5, 40], dtype=np.int32)
    seed = 42
    got = oracle.light_noise(lp, seed, amp, kf)
    t = np.arange(256)
    for i in range(2):
        want = np.zeros(256)
        for f in range(2):
            u0 = (_philox_py((i, f, 1, LGHT), (seed, 0))[0] + 0.5) / 4294967296.0
            want += amp[f] * np.cos(2 * math.pi * kf[f] * t / 256 + 2 * math.pi * u0)
        assert np.allclose(got[i], want, atol=1e-12)
        assert (got[i] ** 2).mean() == pytest.approx((9.0 + 0.25) / 2, rel=1e-9)
    assert not np.allclose(got[0], got[1])


def test_light_chain_conserves_light():
    """The whole chain on configs[0] with the synthetic light LUT: photoelectrons per sensor are conserved from eq. (4.2)
    to the time profile (all of it lands inside the waveform), the scintillation convolution keeps sum(w) of it up to the
    part cut off at the end of the waveform, and the noise-free ADC waveform integrates to G_i x the observed photoelectrons."""
    wl = W.make_config(0)
    ls = W.light_setup(wl, n_det=6)
    _, ne = oracle.quench(wl.params, wl.segments)
    r = oracle.light_chain(ls.params, ls, wl.segments, ne, 7)
    assert np.all(r["vox"] >= 0)
    assert np.allclose(r["ipe"].sum(axis=1), r["npe"].sum(axis=1), rtol=1e-6)
    w = oracle.light_scint_weights(ls.params)
    assert np.all(r["isc"].sum(axis=1) <= r["ipe"].sum(axis=1) * w.sum() * (1 + 1e-12))
    assert np.all(r["isc"].sum(axis=1) >= r["ipe"].sum(axis=1) * 0.97)
    assert np.allclose(r["v"].sum(axis=1), ls.gain * r["nobs"].sum(axis=1) * ls.resp.sum(), rtol=1e-5)
