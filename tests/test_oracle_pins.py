"""Pins of the fp64 CPU oracle against what the paper and the mathematics fix (no GPU).

Each test names the passage of arXiv 2212.09807 (P:L### = /root/reference/PAPER.md line) or the
SURVEY.md 8(c.4) row it checks.  None of them retypes the oracle's own formula: they use printed
values (tests/golden/), invariants, closed forms of special cases, brute force and a per-electron
Monte Carlo written independently in numpy.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2212_09807_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.split("#")[0].strip()
        if line:
            out.append(line.split())
    return out


def _one_segment(xs, ys, zs, xe, ye, ze, dE, ts=0.0, te=0.0):
    f = lambda v: np.atleast_1d(np.asarray(v, dtype=np.float32))
    return dict(xs=f(xs), ys=f(ys), zs=f(zs), ts=f(ts), xe=f(xe), ye=f(ye), ze=f(ze), te=f(te), dE=f(dE))


def _small_setup(nx=12, ny=12, drift=12.0, n_ticks=None, **over):
    p = W.default_params(**over)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, drift, nx, ny, 0)]
    p["n_readout_ticks"] = n_ticks if n_ticks is not None else W._n_ticks(p, drift, 0.0)
    return p, tpcs, W.pad_response_lut(p)


def _chain(p, tpcs, seg):
    dedx, ne = oracle.quench(p, seg)
    dr = oracle.drift(p, tpcs, seg, ne)
    pm = oracle.pixmap(p, tpcs, seg, dr)
    return dedx, ne, dr, pm


# ------------------------------------------------------------------ O1 recombination

def test_recombination_golden_values():
    """SURVEY 8(c.4) O1 table; the paper prints 'around 0.7' for a MIP with both models."""
    for row in _rows("recombination.txt"):
        q, box212, box207, birks = map(float, row)
        seg = _one_segment(0, 0, 5, 0.1, 0, 5, q * 0.1)
        # float32 rounding of 0.1 and dE: use the actual length and energy the oracle sees
        L = float(seg["xe"][0]) - float(seg["xs"][0])
        Q0 = float(seg["dE"][0]) / 23.6e-6
        for model, beta, want in ((1, 0.212, box212), (1, 0.207, box207), (0, 0.212, birks)):
            p = W.default_params(recomb_model=model, box_beta=beta)
            dedx, ne = oracle.quench(p, seg)
            assert dedx[0] == pytest.approx(float(seg["dE"][0]) / L, rel=1e-12)
            assert ne[0] / Q0 == pytest.approx(want, abs=2e-6)
    # 1 mm MIP segment: Q_0 = 8898.31 e-, 6266.62 (Box .212) / 6201.38 (Birks)
    seg = _one_segment(0, 0, 5, 0.1, 0, 5, 0.21)
    assert oracle.quench(W.default_params(recomb_model=1), seg)[1][0] == pytest.approx(6266.62, rel=2e-6)
    assert oracle.quench(W.default_params(recomb_model=0), seg)[1][0] == pytest.approx(6201.38, rel=2e-6)
    for model in (0, 1):                                    # "around 0.7"
        ne = oracle.quench(W.default_params(recomb_model=model, box_beta=0.207), seg)[1][0]
        assert abs(ne / (0.21 / 23.6e-6) - 0.7) < 0.01


def test_recombination_invariants():
    """Birks: 1/R is linear in dE/dx with slope k_b/(A_b eps) and R(0+) = A_b (eq. 3.1).
    Box: R*xi = ln(alpha + xi) so exp(R*xi) - xi = alpha for every dE/dx (eq. 3.2); clamp below ~0.228 (D6)."""
    q = np.array([0.5, 1.0, 2.0, 4.0, 8.0, 16.0, 40.0])
    seg = _one_segment(np.zeros(7), np.zeros(7), np.full(7, 5.0), np.full(7, 0.25), np.zeros(7), np.full(7, 5.0),
                       q * 0.25)
    Q0 = seg["dE"].astype(np.float64) / 23.6e-6
    qd = seg["dE"].astype(np.float64) / 0.25
    eps = 0.5 * 1.38
    R = oracle.quench(W.default_params(recomb_model=0), seg)[1] / Q0
    slope = np.diff(1.0 / R) / np.diff(qd)
    assert np.allclose(slope, 0.0486 / (0.800 * eps), rtol=1e-9)
    assert np.allclose(1.0 / R - slope[0] * qd, 1.0 / 0.800, rtol=1e-9)
    R = oracle.quench(W.default_params(recomb_model=1, box_beta=0.212), seg)[1] / Q0
    xi = 0.212 * qd / eps
    assert np.allclose(np.exp(R * xi) - xi, 0.93, rtol=1e-9)
    assert np.all(np.diff(R[qd >= 2.0]) < 0)                  # falls with dE/dx above a MIP; 'inadequate' below
    low = _one_segment(0, 0, 5, 1.0, 0, 5, 0.2)             # dE/dx = 0.2 < 0.228 -> negative log -> clamp
    assert oracle.quench(W.default_params(recomb_model=1), low)[1][0] == 0.0
    zero = _one_segment(1, 1, 5, 1, 1, 5, 0.2)              # zero length
    assert oracle.quench(W.default_params(), zero)[1][0] == 0.0


# ------------------------------------------------------------------ O2 transport

def test_transport_golden_values():
    """exp(-t/tau) and sigma = sqrt(2 D t) (eqs. 3.3-3.5)."""
    p, tpcs, _ = _small_setup(drift=60.0)
    for row in _rows("transport.txt"):
        d, att, sT_mm, sL_mm, st_ticks = map(float, row)
        seg = _one_segment(2.0, 2.0, d, 2.0, 2.1, d, 0.21)
        ne = np.array([1000.0])
        dr = oracle.drift(p, tpcs, seg, ne)
        assert dr["tpc"][0] == 0
        assert dr["q_a"][0] / 1000.0 == pytest.approx(att, abs=1e-6)
        assert dr["sigma_T"][0] * 10 == pytest.approx(sT_mm, abs=1e-5)
        assert dr["sigma_t"][0] * p["v_drift_cm_us"] * 10 == pytest.approx(sL_mm, abs=1e-5)
        assert dr["sigma_t"][0] / p["tick_us"] == pytest.approx(st_ticks, abs=1e-4)
        assert dr["T_s"][0] == pytest.approx(d / 0.16, rel=1e-7)
    # sigma^2 is linear in drift time, ratio D_T/D_L = 2.2 (eq. 3.5)
    assert (dr["sigma_T"][0] / (dr["sigma_t"][0] * 0.16)) ** 2 == pytest.approx(8.8 / 4.0, rel=1e-12)


def test_drift_two_sided_module_and_inactive():
    """Two TPCs back to back: the sign of eq. (3.3) flips; midpoint outside every TPC -> inactive (D8)."""
    p = W.default_params()
    tpcs = [W.make_tpc(0, 0, -30.0, +1, 30.0, 10, 10, 0), W.make_tpc(0, 0, +30.0, -1, 30.0, 10, 10, 100)]
    seg = _one_segment([1, 1, 1, 50], [1, 1, 1, 1], [-20.0, 20.0, -31.0, 0.0], [1.1, 1.1, 1.1, 50.1], [1, 1, 1, 1],
                       [-20.0, 20.0, -31.0, 0.0], [0.2] * 4, ts=[3.0] * 4, te=[3.0] * 4)
    dr = oracle.drift(p, tpcs, seg, np.full(4, 100.0))
    assert dr["tpc"].tolist() == [0, 1, -1, -1]
    assert dr["T_s"][0] == pytest.approx(3.0 + 10.0 / 0.16)
    assert dr["T_s"][1] == pytest.approx(3.0 + 10.0 / 0.16)
    assert dr["q_a"][2] == 0.0 and dr["q_a"][3] == 0.0
    assert dr["q_a"][0] == pytest.approx(100.0 * math.exp(-(10.0 / 0.16) / 2200.0), rel=1e-12)


# ------------------------------------------------------------------ O3 pixel mapping

def test_pixmap_hand_cases():
    """segment inside one pixel, sigma = 0, W = 5 -> exactly 5x5; clipping at the plane edge."""
    p, tpcs, _ = _small_setup(nx=12, ny=12)
    pitch = p["pixel_pitch_cm"]
    seg = _one_segment((5 + 0.33) * pitch, (6 + 0.44) * pitch, 0.0, (5 + 0.68) * pitch, (6 + 0.55) * pitch, 0.0, 0.1)
    _, _, dr, pm = _chain(p, tpcs, seg)
    assert (pm["ix0"][0], pm["ix1"][0], pm["iy0"][0], pm["iy1"][0]) == (3, 7, 4, 8)
    assert pm["npix"][0] == 25 and pm["a_lo"][0] == 53 and pm["a_hi"][0] == 56
    assert pm["jt0"][0] == 0 and pm["jt1"][0] == 0
    seg = _one_segment(0.2 * pitch, 0.5 * pitch, 0.0, 0.4 * pitch, 0.5 * pitch, 0.0, 0.1)   # corner pixel
    _, _, dr, pm = _chain(p, tpcs, seg)
    assert (pm["ix0"][0], pm["ix1"][0], pm["iy0"][0], pm["iy1"][0]) == (0, 2, 0, 2) and pm["npix"][0] == 9
    # sample count N = max(1, ceil(L / 10 um))
    seg = _one_segment(1.0, 1.0, 1.0, 1.0 + 0.0255, 1.0, 1.0, 0.1)
    assert _chain(p, tpcs, seg)[3]["n_samples"][0] == 26
    seg = _one_segment(1.0, 1.0, 1.0, 1.0 + 1e-5, 1.0, 1.0, 0.1)
    assert _chain(p, tpcs, seg)[3]["n_samples"][0] == 1


def test_pixmap_complete_and_minimal():
    """Every pixel that receives more than 1e-5 of a segment's charge lies in its rectangle (completeness,
    the 5-sigma tail bound of SURVEY 8(c.1) O3), and for an axis-aligned segment the charged range is the
    exact set of pixels within reach (minimality)."""
    p, tpcs, lut = _small_setup(nx=14, ny=14, drift=12.0)
    rng = np.random.Generator(np.random.PCG64(5))
    pitch = p["pixel_pitch_cm"]
    for trial in range(3):
        c = np.array([rng.uniform(5, 9) * pitch, rng.uniform(5, 9) * pitch, rng.uniform(0.5, 11.0)])
        d = W._iso_dir(rng)
        seg = _one_segment(*(c - 0.05 * d), *(c + 0.05 * d), 0.21)
        _, _, dr, pm = _chain(p, tpcs, seg)
        ix, iy = np.meshgrid(np.arange(14), np.arange(14))
        waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, ix.ravel(), iy.ravel())
        amp = np.abs(waves).sum(axis=1).reshape(14, 14)
        inside = np.zeros((14, 14), bool)
        inside[pm["iy0"][0]:pm["iy1"][0] + 1, pm["ix0"][0]:pm["ix1"][0] + 1] = True
        assert amp[~inside].max() < 1e-5 * dr["q_a"][0]
        assert amp[inside].min() > 0.0
    # axis-aligned along x, sigma_T known: charged pixels = those within 5 sigma of [u_s, u_e]
    seg = _one_segment(6.25 * pitch, 7.5 * pitch, 8.0, 6.75 * pitch, 7.5 * pitch, 8.0, 0.21)
    _, _, dr, pm = _chain(p, tpcs, seg)
    r = 5.0 * dr["sigma_T"][0]
    lo = math.floor((float(seg["xs"][0]) - r) / pitch)
    hi = math.floor((float(seg["xe"][0]) + r) / pitch)
    assert pm["ix0"][0] == lo - 2 and pm["ix1"][0] == hi + 2


# ------------------------------------------------------------------ O4 induced current

def test_point_charge_reproduces_lut():
    """zero diffusion, L -> 0 (N = 1), above a bin centre: the waveform on every pixel of
    the window is Q_a times the LUT series of the bin it is seen through, shifted to the arrival tick."""
    p, tpcs, lut = _small_setup(nx=9, ny=9, drift=5.0, n_ticks=260)
    pitch, nb = p["pixel_pitch_cm"], p["bins_per_pixel"]
    binw = pitch / nb
    ca, cb = 3, 7                                          # in-pixel bin of the charge, pixel (4, 4)
    x = 4 * pitch + (ca + 0.5) * binw
    y = 4 * pitch + (cb + 0.5) * binw
    seg = _one_segment(x, y, 0.0, x + 2e-6, y, 0.0, 0.21, ts=1.23, te=1.23)   # at the anode: sigma = 0
    _, ne, dr, pm = _chain(p, tpcs, seg)
    assert dr["sigma_T"][0] == 0.0 and pm["n_samples"][0] == 1
    j = int(math.floor(1.23 / 0.1))
    K = p["lut_ticks"]
    for (ix, iy) in [(4, 4), (3, 4), (4, 6), (2, 2), (6, 5)]:
        waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [ix], [iy])
        cx = ca + nb * (4 - ix + 2)
        cy = cb + nb * (4 - iy + 2)
        want = np.zeros(p["n_readout_ticks"])
        want[j:j + K] = dr["q_a"][0] * lut[cy, cx].astype(np.float64)
        assert np.allclose(waves[0], want, rtol=1e-13, atol=1e-12)
    waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [4, 3], [4, 4])
    assert qp[0] == pytest.approx(dr["q_a"][0], rel=1e-6)   # LUT normalised to one electron
    assert abs(qp[1]) < 1e-5 * dr["q_a"][0]                  # neighbours: bipolar, integrates to zero


def test_charge_conservation_and_linearity():
    """sum over pixels and ticks of I equals sum of Q_a for tracks >= 2 pixels from the
    edge (harness LUT columns sum to 1/0); the result is linear in the segments and invariant under
    translation by whole pixels and whole ticks."""
    p, tpcs, lut = _small_setup(nx=14, ny=14, drift=12.0, n_ticks=1100)
    rng = np.random.Generator(np.random.PCG64(11))
    pitch = p["pixel_pitch_cm"]
    c = np.array([6.3 * pitch, 7.1 * pitch, 6.0])
    d = np.array([0.6, 0.3, 0.74])
    d /= np.linalg.norm(d)
    seg = W.line_segments(c - 0.15 * d, c + 0.15 * d, 0.1, 2.0, lambda s, L, n: np.array([2.1, 6.0, 3.0]))
    _, _, dr, pm = _chain(p, tpcs, seg)
    ix, iy = oracle.active_pixels(tpcs, pm, dr, 0)
    waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, ix, iy)
    assert qp.sum() == pytest.approx(dr["q_a"].sum(), rel=2e-6)
    # linearity: sum of single-segment results
    acc = np.zeros_like(waves)
    for s in range(3):
        one = {k: v[s:s + 1] for k, v in seg.items()}
        _, _, dr1, pm1 = _chain(p, tpcs, one)
        acc += oracle.pixel_currents(p, tpcs, lut, dr1, pm1, 0, ix, iy)[0]
    assert np.allclose(acc, waves, rtol=1e-12, atol=1e-9)
    # translation by (+2, -1) pixels and +7 ticks
    seg2 = {k: v.copy() for k, v in seg.items()}
    # shift in float64 then round: the shifted float32 coordinates differ from the exact shift by < 1e-6 cm
    for k in ("xs", "xe"):
        seg2[k] = (seg[k].astype(np.float64) + 2 * pitch).astype(np.float32)
    for k in ("ys", "ye"):
        seg2[k] = (seg[k].astype(np.float64) - 1 * pitch).astype(np.float32)
    for k in ("ts", "te"):
        seg2[k] = (seg[k].astype(np.float64) + 0.7).astype(np.float32)
    _, _, dr2, pm2 = _chain(p, tpcs, seg2)
    waves2, _ = oracle.pixel_currents(p, tpcs, lut, dr2, pm2, 0, ix + 2, iy - 1)
    scale = np.abs(waves).max()
    assert np.abs(waves2[:, 7:] - waves[:, :-7]).max() < 2e-4 * scale   # float32 rounding of the shifted inputs


def test_long_track_closed_form():
    """a long straight track parallel to the plane, centred on a pixel row, deposits
    Q_p = lambda * pitch * erf(pitch / (2 sqrt(2) sigma_T)) on each pixel of that row."""
    p, tpcs, lut = _small_setup(nx=16, ny=9, drift=12.0, n_ticks=1000)
    pitch = p["pixel_pitch_cm"]
    y = 4.5 * pitch
    seg = W.line_segments([1.0 * pitch, y, 10.0], [15.0 * pitch, y, 10.0], 0.1, 0.0, lambda s, L, n: np.full(n, 2.1))
    _, _, dr, pm = _chain(p, tpcs, seg)
    lam = dr["q_a"].sum() / (14.0 * pitch)
    sT = dr["sigma_T"][0]
    waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [7, 8, 7], [4, 4, 5])
    want_row = lam * pitch * math.erf(pitch / (2.0 * math.sqrt(2.0) * sT))
    assert qp[0] == pytest.approx(want_row, rel=2e-5)
    assert qp[1] == pytest.approx(want_row, rel=2e-5)
    want_next = lam * pitch * 0.5 * (math.erf(1.5 * pitch / (math.sqrt(2.0) * sT)) - math.erf(0.5 * pitch / (math.sqrt(2.0) * sT)))
    assert qp[2] == pytest.approx(want_next, rel=2e-4, abs=0.05)
    # whole chain: MIP at 10 cm -> 6.091e4 e-/cm
    assert lam == pytest.approx(2.1 / 23.6e-6 * 0.704248 * 0.971991, rel=1e-4)


def test_direct_sum_equals_lattice_form():
    """The literal six-fold sum of SURVEY 8(c.1) equals the two-step (rho on the lattice, then eq. 3.7) form."""
    p, tpcs, lut = _small_setup(nx=7, ny=7, drift=3.0, n_ticks=150, lut_ticks=40, window_pixels=3,
                                sample_step_cm=0.01)
    pitch = p["pixel_pitch_cm"]
    seg = _one_segment([3.2 * pitch, 3.6 * pitch], [3.4 * pitch, 2.9 * pitch], [1.0, 0.0],
                       [3.35 * pitch, 3.7 * pitch], [3.5 * pitch, 2.95 * pitch], [1.05, 0.0], [0.1, 0.05])
    _, _, dr, pm = _chain(p, tpcs, seg)
    for (ix, iy) in [(3, 3), (2, 3), (4, 2)]:
        a = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [ix], [iy])[0][0]
        b = oracle.direct_current(p, lut, dr, pm, 0, ix, iy)
        assert np.abs(a).max() > 0
        assert np.allclose(a, b, rtol=1e-11, atol=1e-12 * np.abs(a).max())


def test_per_electron_monte_carlo():
    """SURVEY 8(c.4) O4(iv) / BASELINE north_star: brute-force per-electron Monte Carlo of eqs. (3.8)-(3.9):
    every electron is placed at one of the N points, displaced by N(0, sigma_T) in x and y and N(0, sigma_L)
    along the drift, looked up in the nearest LUT bin at its arrival tick.  The mean agrees with the oracle's
    expectation form within 5 standard errors per (pixel, tick)."""
    p, tpcs, lut = _small_setup(nx=9, ny=9, drift=12.0, n_ticks=620)
    pitch, nb, K, dt = p["pixel_pitch_cm"], p["bins_per_pixel"], p["lut_ticks"], p["tick_us"]
    binw = pitch / nb
    c = np.array([4.4 * pitch, 4.7 * pitch, 4.0])
    d = np.array([0.5, -0.4, 0.77])
    d /= np.linalg.norm(d)
    seg = W.line_segments(c - 0.1 * d, c + 0.1 * d, 0.1, 0.5, lambda s, L, n: np.array([2.1, 4.0]))
    _, _, dr, pm = _chain(p, tpcs, seg)
    pix = [(4, 4), (5, 4), (4, 5), (3, 3)]
    waves, qp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [a for a, _ in pix], [b for _, b in pix])
    rng = np.random.Generator(np.random.PCG64(99))
    nbatch, per = 16, 60000
    nt = p["n_readout_ticks"]
    est = np.zeros((nbatch, len(pix), nt))
    lut64 = lut.astype(np.float64)
    for bi in range(nbatch):
        for s in range(2):
            N = int(pm["n_samples"][s])
            mu = rng.integers(0, N, size=per)
            f = (mu + 0.5) / N
            x = dr["u_s"][s] + (dr["u_e"][s] - dr["u_s"][s]) * f + rng.normal(0, dr["sigma_T"][s], per)
            y = dr["v_s"][s] + (dr["v_e"][s] - dr["v_s"][s]) * f + rng.normal(0, dr["sigma_T"][s], per)
            T = dr["T_s"][s] + (dr["T_e"][s] - dr["T_s"][s]) * f + rng.normal(0, dr["sigma_t"][s], per)
            a = np.floor(x / binw).astype(int)
            b = np.floor(y / binw).astype(int)
            j = np.floor((T - p["t_origin_us"]) / dt).astype(int)
            w = dr["q_a"][s] / per
            for k, (ix, iy) in enumerate(pix):
                cx, cy = a - nb * (ix - 2), b - nb * (iy - 2)
                ok = (cx >= 0) & (cx < 5 * nb) & (cy >= 0) & (cy < 5 * nb) & (j >= 0) & (j <= nt - K)
                cell = (cy[ok] * 5 * nb + cx[ok]) * (nt - K + 1) + j[ok]
                G = np.bincount(cell, minlength=(5 * nb) ** 2 * (nt - K + 1)).reshape((5 * nb) ** 2, nt - K + 1)
                rows = np.nonzero(G.any(axis=1))[0]
                for r in rows:
                    cols = np.nonzero(G[r])[0]
                    for jj in cols:
                        est[bi, k, jj:jj + K] += w * G[r, jj] * lut64.reshape(-1, K)[r]
    mean = est.mean(axis=0)
    se = est.std(axis=0, ddof=1) / math.sqrt(nbatch)
    big = np.abs(waves) > 1e-3 * np.abs(waves).max()
    zscore = np.abs(mean - waves)[big] / np.maximum(se[big], 1e-9)
    assert big.sum() > 200
    assert np.quantile(zscore, 0.99) < 4.0 and zscore.max() < 6.0
    # integrated charge per pixel agrees to MC precision as well
    q_mc = est.sum(axis=2)
    q_se = q_mc.std(axis=0, ddof=1) / math.sqrt(nbatch)
    # (tails holding < 1e-6 of the charge are invisible to 1e6 electrons)
    assert np.all(np.abs(q_mc.mean(axis=0) - qp) < 5 * q_se + 1e-6 * dr["q_a"].sum())


# ------------------------------------------------------------------ O6 electronics + Philox

def test_philox_known_answers():
    """Philox4x32-10 known-answer vectors (tests/golden/philox4x32_10.txt)."""
    for row in _rows("philox4x32_10.txt"):
        h = [int(x, 16) for x in row]
        assert oracle.philox4x32_10(h[:4], h[4:6]) == h[6:]


def test_noise_normal_moments():
    """Box-Muller normals keyed by (seed, pixel, tick): mean 0, variance 1, fourth moment 3, uncorrelated."""
    z = np.array([oracle.noise_normals(1234, pix, t) for pix in range(40) for t in range(500)])
    n = z.shape[0]
    for k in range(3):
        assert abs(z[:, k].mean()) < 4 / math.sqrt(n)
        assert abs(z[:, k].var() - 1) < 4 * math.sqrt(2 / n)
        assert abs((z[:, k] ** 4).mean() - 3) < 4 * math.sqrt(96 / n)
    assert abs(np.corrcoef(z.T)[0, 1]) < 4 / math.sqrt(n) and abs(np.corrcoef(z.T)[0, 2]) < 4 / math.sqrt(n)
    assert oracle.noise_normals(1234, 7, 9) != oracle.noise_normals(1235, 7, 9)


def test_electronics_hand_cases():
    """constant current c e-/tick without noise crosses 7000 e- at tick ceil(7000/c) - 1, is
    sampled 16 ticks (1.6 us) later with adc = floor((580 + 4 q/1000 - 288) / 3.953125); a pixel that
    never reaches the threshold gives no hit; 28 mV <=> 7000 e- at 4 mV/ke- (P:L708)."""
    p = W.default_params(n_readout_ticks=400)
    lsb = (1300.0 - 288.0) / 256
    assert lsb == 3.953125
    for c in (250.0, 999.0, 3500.0, 7000.0):
        wave = np.full((1, 400), c)
        hp, ht, ha, cnt = oracle.electronics(p, 0, [17], wave)
        n_c = math.ceil(7000.0 / c) - 1
        assert ht[0] == n_c + 16
        q_s = c * (n_c + 17)
        assert ha[0] == min(255, math.floor((580 + 4 * q_s / 1000 - 288) / lsb))
        # after the reset the same pattern repeats with period (n_c + 17) ticks
        assert np.all(np.diff(ht) == n_c + 17)
        assert cnt[0] == len(ht) == (400 // (n_c + 17))
    sub = np.zeros((1, 400))
    sub[0, 10:60] = 139.0                                    # 6950 e- in total: below threshold
    assert oracle.electronics(p, 0, [3], sub)[3][0] == 0
    edge = np.zeros((1, 400))
    edge[0, 100] = 7000.0                                    # exactly the threshold: q >= threshold fires (D13)
    hp, ht, ha, cnt = oracle.electronics(p, 0, [3], edge)
    assert ht.tolist() == [116] and ha[0] == math.floor((580 + 28.0 - 288) / lsb)
    late = np.zeros((1, 400))
    late[0, 390] = 9000.0                                    # sample tick 406 is past the window: nothing (O6 step 4)
    assert oracle.electronics(p, 0, [3], late)[3][0] == 0
    # whole chain estimate of SURVEY 8(c.4): 2.70e4 e- collected in one hit -> ADC about 101
    one = np.zeros((1, 400))
    one[0, 50:60] = 2700.0
    assert abs(int(oracle.electronics(p, 0, [3], one)[2][0]) - 101) <= 1


def test_electronics_noise_is_keyed_and_reproducible():
    """Noise terms: reset / discriminator / uncorrelated; draws depend only on (seed, pixel, tick)."""
    p = W.default_params(n_readout_ticks=300, noise_reset_e=900.0, noise_uncorr_e=500.0, noise_disc_e=650.0)
    wave = np.zeros((2, 300))
    wave[:, 20:80] = 400.0
    a = oracle.electronics(p, 42, [5, 6], wave)
    b = oracle.electronics(p, 42, [5, 6], wave)
    c = oracle.electronics(p, 43, [5, 6], wave)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    assert not all(np.array_equal(x, y) for x, y in zip(a, c))
    # uncorrelated noise alone shifts the ADC by (500 e- * z_u) * 4 mV/ke- / LSB counts at the sample tick
    p2 = W.default_params(n_readout_ticks=300, noise_uncorr_e=500.0)
    hp, ht, ha, _ = oracle.electronics(p2, 42, [5], wave[:1])
    z = oracle.noise_normals(42, 5, int(ht[0]))
    q = 400.0 * (ht[0] - 20 + 1)
    assert ha[0] == math.floor((580 + 4 * (q + 500.0 * z[1]) / 1000 - 288) / 3.953125)


# ---- the four noise / timing branches of O6, each against values worked out HERE from the Philox words -----------------
# (an independent pure-Python Philox4x32-10 + Box-Muller: nothing below calls the oracle's own normals)

def _philox_py(ctr, key):
    """Philox4x32-10 as published (Salmon et al., SC'11): 10 rounds of two 32x32 -> 64 multiplies, key bumped by the
    Weyl constants each round."""
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    M = 0xFFFFFFFF
    for _ in range(10):
        p0, p1 = 0xD2511F53 * c0, 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M, p1 & M, ((p0 >> 32) ^ c3 ^ k1) & M, p0 & M
        k0, k1 = (k0 + 0x9E3779B9) & M, (k1 + 0xBB67AE85) & M
    return [c0, c1, c2, c3]


def _normals_py(seed, pixel, tick):
    """(z_d, z_u, z_r) of SURVEY 8(c.1) O6 / reading D16: counter (pixel, tick, 0, 0), key (seed lo, seed hi),
    u_i = (x_i + 0.5) 2^-32, z_d = r01 cos, z_u = r01 sin (pair u0, u1), z_r = r23 cos (pair u2, u3)."""
    x = _philox_py((pixel, tick, 0, 0), (seed & 0xFFFFFFFF, seed >> 32))
    u = [(xi + 0.5) / 4294967296.0 for xi in x]
    r01, r23 = math.sqrt(-2 * math.log(u[0])), math.sqrt(-2 * math.log(u[2]))
    return r01 * math.cos(2 * math.pi * u[1]), r01 * math.sin(2 * math.pi * u[1]), r23 * math.cos(2 * math.pi * u[3])


def _adc(q_s):
    return min(255, max(0, math.floor((580 + 4 * q_s / 1000 - 288) / 3.953125)))


def test_python_philox_matches_the_published_vectors():
    """The test's own generator against the Random123 known-answer vectors (tests/golden/philox4x32_10.txt), and the
    oracle's normals against the test's for a spread of (seed, pixel, tick): both sides of every pin below are anchored."""
    for row in _rows("philox4x32_10.txt"):
        h = [int(x, 16) for x in row]
        assert _philox_py(h[:4], h[4:6]) == h[6:]
    for seed, pix, tick in ((0, 0, 0), (42, 5, 117), (2 ** 40 + 17, 10 ** 7, 3400), (0x22120983, 123456, 1)):
        assert np.allclose(oracle.noise_normals(seed, pix, tick), _normals_py(seed, pix, tick), rtol=1e-13, atol=1e-15)


def test_electronics_reset_noise_branch():
    """P:L710 "random pedestal shift after every trigger reset" (reading D16: q = 900 z_r(pixel, sample tick) after the
    reset, z_r from the SECOND Box-Muller pair).  Constant 1000 e-/tick: the first hit is noise-free (crossing at tick 6,
    sample at 22, q_s = 23000); the second crossing is the first tick n > 22 with 900 z_r + 1000 (n - 22) >= 7000, its
    sample 16 ticks later holds 900 z_r + 1000 (n_s - 22).  A reset that used z_d or z_u, or that was applied before the
    sample was taken, or a q that kept the collected charge, gives other ticks / counts on these pixels."""
    p = W.default_params(n_readout_ticks=120, noise_reset_e=900.0)
    seed = 20221209
    moved = other_z = 0
    for pid in range(40, 64):
        hp, ht, ha, cnt = oracle.electronics(p, seed, [pid], np.full((1, 120), 1000.0))
        zd, zu, zr = _normals_py(seed, pid, 22)
        q0 = 900.0 * zr
        n_c2 = 22 + math.ceil((7000.0 - q0) / 1000.0)
        assert ht[0] == 22 and ha[0] == _adc(23000.0)
        assert ht[1] == n_c2 + 16 and ha[1] == _adc(q0 + 1000.0 * (n_c2 + 16 - 22))
        zr2 = _normals_py(seed, pid, n_c2 + 16)[2]                 # and once more: third hit from the second reset
        n_c3 = n_c2 + 16 + math.ceil((7000.0 - 900.0 * zr2) / 1000.0)
        assert ht[2] == n_c3 + 16 and ha[2] == _adc(900.0 * zr2 + 1000.0 * (n_c3 - n_c2))
        moved += (n_c2 != 29) or _adc(q0 + 1000.0 * (n_c2 - 6)) != _adc(23000.0)
        for zalt in (zd, zu):
            alt = 22 + math.ceil((7000.0 - 900.0 * zalt) / 1000.0)
            other_z += (alt != n_c2) or _adc(900.0 * zalt + 1000.0 * (alt - 6)) != ha[1]
    assert moved >= 12 and other_z >= 24          # the draws do move the result, and the wrong normal would not pass


def test_electronics_uncorrelated_noise_branch():
    """P:L710 uncorrelated noise 500 e- (reading D16: added to the SAMPLED value only, z_u = second normal of the first
    Box-Muller pair of the (pixel, sample tick) draw; the integrated charge itself is untouched, so the timing is the
    noise-free one).  400 e-/tick from tick 20: crossing at 37, sample at 53 with 13600 e- + 500 z_u."""
    p = W.default_params(n_readout_ticks=120, noise_uncorr_e=500.0)
    wave = np.zeros((1, 120))
    wave[0, 20:80] = 400.0
    seed, differs = 31337, 0
    for pid in range(200, 240):
        hp, ht, ha, cnt = oracle.electronics(p, seed, [pid], wave)
        zd, zu, zr = _normals_py(seed, pid, 53)
        assert ht[0] == 53 and ha[0] == _adc(13600.0 + 500.0 * zu)
        differs += (_adc(13600.0 + 500.0 * zd) != ha[0]) + (_adc(13600.0 + 500.0 * zr) != ha[0]) + (_adc(13600.0) != ha[0])
        # second hit: the reset left no charge (reset noise off), 26 more ticks of 400 e- remain: 10400 e- >= 7000 at tick 71
        assert ht[1] == 71 + 16 and ha[1] == _adc(10400.0 + 500.0 * _normals_py(seed, pid, 87)[1])
    assert differs >= 15          # (500 e- is half an ADC count: a wrong normal changes about one count in four)


def test_electronics_discriminator_noise_branch():
    """P:L710 discriminator noise 650 e- (reading D16: fresh every tick, on the threshold, z_d = FIRST normal of the
    (pixel, tick) draw).  The charge ramps to 6800 e- in ten ticks and stays there, 200 e- = 0.31 sigma below the
    threshold: the channel fires at the first tick n with q(n) >= 7000 + 650 z_d(pixel, n), taken from the per-tick
    normals worked out here; the sample 16 ticks later reads 6800 e- (no other noise term is on)."""
    p = W.default_params(n_readout_ticks=200, noise_disc_e=650.0)
    wave = np.zeros((1, 200))
    wave[0, :10] = 680.0
    q = np.cumsum(wave[0])
    seed = 777
    late = not_first = 0
    for pid in range(100, 130):
        z = [_normals_py(seed, pid, n) for n in range(200)]
        n_c = next(n for n in range(200) if q[n] >= 7000.0 + 650.0 * z[n][0])
        hp, ht, ha, cnt = oracle.electronics(p, seed, [pid], wave)
        assert ht[0] == n_c + 16 and ha[0] == _adc(q[n_c + 16])
        late += n_c > 9
        alt = [next(n for n in range(200) if q[n] >= 7000.0 + 650.0 * z[n][k]) for k in (1, 2)]
        not_first += (alt[0] != n_c) + (alt[1] != n_c)
        # after the sample the charge is gone (reset, no reset noise): nothing can fire again
        assert cnt[0] == 1
    assert late >= 10 and not_first >= 30          # several ticks "within +-650 z_d of 7000 e-", and z_u / z_r would differ


def test_electronics_periodic_reset_branch():
    """P:L708 "periodic reset" (reading D17: every periodic_reset_ticks an ARMED channel loses its charge, at the START
    of the tick, before that tick's charge is integrated; a channel in its hold is not touched).
    (i) 100 e-/tick crosses 7000 e- at tick 69 without the reset and never with a period of 50 ticks (at most 5000 e-).
    (ii) 1000 e-/tick, period 7: crossing at 6 (7000 e- after ticks 0..6; a reset at tick 7 comes too late), sample 22;
    ticks 23..27 collect 5000, tick 28 resets then adds 1000, ticks 29..34 reach 7000: crossing 34, sample 50; and so
    on every 28 ticks, each sample holding 7000 + 16 x 1000 e-.  A reset applied AFTER the tick's charge would clear
    the 6000 e- of tick 28 to zero and cross at 35."""
    trickle = np.full((1, 400), 100.0)
    assert oracle.electronics(W.default_params(n_readout_ticks=400), 0, [9], trickle)[1].tolist()[0] == 69 + 16
    assert oracle.electronics(W.default_params(n_readout_ticks=400, periodic_reset_ticks=50), 0, [9], trickle)[3][0] == 0
    p = W.default_params(n_readout_ticks=140, periodic_reset_ticks=7)
    hp, ht, ha, cnt = oracle.electronics(p, 0, [9], np.full((1, 140), 1000.0))
    assert ht.tolist() == [22, 50, 78, 106, 134]
    assert ha.tolist() == [_adc(23000.0)] * 5
    # during the hold (ticks 7, 14, 21 fall inside the first one) nothing is cleared: the sample holds all 23 ticks
    assert _adc(23000.0) != _adc(23000.0 - 7000.0)


def test_electronics_min_spacing_branch():
    """consecutive samples are at least min_spacing_ticks apart (1.1 us = 11 ticks in the paper, where the 1.6 us
    hold makes it moot; here 40 > hold + 1).  7000 e-/tick re-crosses at once after every reset, so the spacing is what
    paces the hits: crossing at 0, sample 16; re-armed for a crossing at tick 16 + 40 - 16 = 40 (>=, not >), sample 56;
    then 96, 136.  With the default spacing the same current gives a hit every 17 ticks."""
    wave = np.full((1, 160), 7000.0)
    p = W.default_params(n_readout_ticks=160, min_spacing_ticks=40)
    hp, ht, ha, cnt = oracle.electronics(p, 0, [1], wave)
    assert ht.tolist() == [16, 56, 96, 136]
    # 17 x 7000 e- = 476 mV over the 580 mV pedestal -> count 194; 40 x 7000 e- saturates the 8-bit ADC
    assert ha.tolist() == [194, 255, 255, 255] and _adc(17 * 7000.0) == 194
    # charge keeps integrating while the channel waits to be re-armed: 40 ticks x 7000 e- at every later sample
    p2 = W.default_params(n_readout_ticks=160, min_spacing_ticks=40, gain_mv_per_ke=0.01)
    ha2 = oracle.electronics(p2, 0, [1], wave)[2]
    lsb = (1300.0 - 288.0) / 256
    assert ha2.tolist() == [math.floor((580 + 0.01 * 7 * 17 - 288) / lsb)] + [math.floor((580 + 0.01 * 7 * 40 - 288) / lsb)] * 3
    ht0 = oracle.electronics(W.default_params(n_readout_ticks=160), 0, [1], wave)[1]
    assert ht0.tolist() == list(range(16, 160, 17))


def test_pixmap_tick_range_with_diffusion():
    """O3 tick range and charged-bin box with sigma > 0 (reading D10), numbers worked by hand: one segment at 10 -> 10.05 cm
    of drift, t_mid = 10.025 / 0.16 = 62.65625 us, sigma_L = sqrt(2 x 4e-6 x 62.65625) = 0.0223886 cm -> sigma_t =
    0.1399288 us, 5 sigma_t = 0.699644 us; T_s = 62.5, T_e = 62.8125 us -> jt0 = floor(618.0036) = 618, jt1 =
    floor(635.1214) = 635.  sigma_T = sqrt(2 x 8.8e-6 x 62.65625) = 0.0332077 cm, 5 sigma_T = 0.166038 cm; u from
    2.3 pitch = 1.01982 to 1.04982 cm, bin 0.04434 cm -> a_lo = floor(19.2553) = 19, a_hi = floor(27.4213) = 27."""
    p, tpcs, _ = _small_setup(nx=12, ny=12, drift=12.0)
    pitch = p["pixel_pitch_cm"]
    seg = _one_segment(2.3 * pitch, 5.5 * pitch, 10.0, 2.3 * pitch + 0.03, 5.5 * pitch, 10.05, 0.21)
    _, _, dr, pm = _chain(p, tpcs, seg)
    assert dr["sigma_t"][0] == pytest.approx(0.1399288, rel=1e-6) and dr["sigma_T"][0] == pytest.approx(0.0332077, rel=1e-6)
    assert (pm["jt0"][0], pm["jt1"][0]) == (618, 635)
    assert (pm["a_lo"][0], pm["a_hi"][0]) == (19, 27)
    # v is constant at 5.5 pitch = bin 55.0: +- 0.166038 / 0.04434 = 3.7446 bins -> floor(51.255) .. floor(58.745)
    assert (pm["b_lo"][0], pm["b_hi"][0]) == (51, 58)
    # pixel rectangle: charged pixels 1..2 (x) and 5 (y), widened by H = 2
    assert (pm["ix0"][0], pm["ix1"][0], pm["iy0"][0], pm["iy1"][0]) == (0, 4, 3, 7)
    # t_origin shifts the ticks, not the box: 3.0 us later -> 30 ticks earlier
    p2 = dict(p, t_origin_us=3.0)
    pm2 = oracle.pixmap(p2, tpcs, seg, oracle.drift(p2, tpcs, seg, oracle.quench(p2, seg)[1]))
    assert (pm2["jt0"][0], pm2["jt1"][0]) == (588, 605)


# ------------------------------------------------------------------ O4r eq. (3.9) as printed (random perturbations)
def _random_case():
    p, tpcs, lut = _small_setup(nx=14, ny=14, drift=12.0, n_ticks=1100)
    pitch = p["pixel_pitch_cm"]
    c = np.array([6.3 * pitch, 7.1 * pitch, 6.0])
    d = np.array([0.6, 0.3, 0.74])
    d /= np.linalg.norm(d)
    seg = W.line_segments(c - 0.15 * d, c + 0.15 * d, 0.1, 2.0, lambda s, L, n: np.array([2.1, 6.0, 3.0]))
    _, _, dr, pm = _chain(p, tpcs, seg)
    ix, iy = oracle.active_pixels(tpcs, pm, dr, 0)
    return p, tpcs, lut, dr, pm, ix, iy


def test_random_estimator_conserves_charge_exactly():
    """Eq. (3.9): every perturbed point carries Q_a / (N M) into exactly one LUT cell, and every harness LUT
    series over the centre pixel sums to one electron: the sum over pixels and ticks is sum Q_a whatever the
    draws, for any M and seed."""
    p, tpcs, lut, dr, pm, ix, iy = _random_case()
    for m, seed in ((1, 3), (4, 99), (7, 2 ** 40 + 5)):
        _, qp = oracle.pixel_currents_random(p, tpcs, lut, dr, pm, 0, ix, iy, m, seed)
        assert qp.sum() == pytest.approx(dr["q_a"].sum(), rel=2e-6)


def test_random_estimator_equals_expectation_without_diffusion():
    """sigma = 0 (charge at the anode): the perturbations vanish and eq. (3.9) is the expectation form, term by term."""
    p, tpcs, lut = _small_setup(nx=9, ny=9, drift=5.0, n_ticks=260)
    pitch = p["pixel_pitch_cm"]
    seg = W.line_segments([3.2 * pitch, 4.1 * pitch, 0.0], [4.9 * pitch, 4.6 * pitch, 0.0], 0.1, 0.7, W._mip(2.1))
    _, _, dr, pm = _chain(p, tpcs, seg)
    assert np.all(dr["sigma_T"] == 0.0)
    ix, iy = oracle.active_pixels(tpcs, pm, dr, 0)
    w0, q0 = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, ix, iy)
    w1, q1 = oracle.pixel_currents_random(p, tpcs, lut, dr, pm, 0, ix, iy, 3, 12345)
    assert np.allclose(w1, w0, rtol=1e-12, atol=1e-9 * np.abs(w0).max())


def test_random_estimator_one_point_by_hand():
    """One segment with N = 1, M = 1: the single perturbed point, placed here with numpy from the Philox words
    (counter (s, mu, nu, 'RAND'), key = seed; Box-Muller; reading D25), decides the one LUT cell that gets Q_a."""
    p, tpcs, lut = _small_setup(nx=9, ny=9, drift=8.0, n_ticks=800)
    pitch, nb, K = p["pixel_pitch_cm"], p["bins_per_pixel"], p["lut_ticks"]
    x, y, z = 4.37 * pitch, 4.61 * pitch, 5.0
    seg = _one_segment(x, y, z, x + 4e-4, y, z, 0.21, ts=0.4, te=0.4)
    _, _, dr, pm = _chain(p, tpcs, seg)
    assert pm["n_samples"][0] == 1 and dr["sigma_T"][0] > 0
    seed = 0x1234ABCD5678
    xw = oracle.philox4x32_10((0, 0, 0, 0x52414E44), (seed & 0xFFFFFFFF, seed >> 32))
    u = (np.array(xw, dtype=np.float64) + 0.5) / 4294967296.0
    r01, r23 = math.sqrt(-2 * math.log(u[0])), math.sqrt(-2 * math.log(u[2]))
    z1, z2, z3 = r01 * math.cos(2 * math.pi * u[1]), r01 * math.sin(2 * math.pi * u[1]), r23 * math.cos(2 * math.pi * u[3])
    assert np.allclose(oracle.perturbation_normals(seed, 0, 0, 0, 5.0), [z1, z2, z3], rtol=1e-14)
    um = 0.5 * (dr["u_s"][0] + dr["u_e"][0]) + dr["sigma_T"][0] * z1
    vm = 0.5 * (dr["v_s"][0] + dr["v_e"][0]) + dr["sigma_T"][0] * z2
    Tm = 0.5 * (dr["T_s"][0] + dr["T_e"][0]) + dr["sigma_t"][0] * z3
    binw = pitch / nb
    a, b, j = int(math.floor(um / binw)), int(math.floor(vm / binw)), int(math.floor(Tm / p["tick_us"]))
    pix_x, pix_y = a // nb, b // nb
    for (ix, iy) in [(pix_x, pix_y), (pix_x + 1, pix_y), (pix_x - 1, pix_y + 2)]:
        waves, _ = oracle.pixel_currents_random(p, tpcs, lut, dr, pm, 0, [ix], [iy], 1, seed)
        cx, cy = a - nb * (ix - 2), b - nb * (iy - 2)
        want = np.zeros(p["n_readout_ticks"])
        want[j:j + K] = dr["q_a"][0] * lut[cy, cx].astype(np.float64)
        assert np.allclose(waves[0], want, rtol=1e-13, atol=1e-12)
    # the clamp of reading D25
    assert np.all(np.abs(oracle.perturbation_normals(seed, 0, 0, 0, 0.25)) <= 0.25)


def test_random_estimator_is_unbiased():
    """the M perturbations estimate the diffusion integral; their mean over independent seeds converges to
    the expectation form (reading D1) within 5 standard errors on every pixel carrying charge."""
    p, tpcs, lut, dr, pm, ix, iy = _random_case()
    _, q_exp = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, ix, iy)
    runs = np.array([oracle.pixel_currents_random(p, tpcs, lut, dr, pm, 0, ix, iy, 2, 1000 + k)[1] for k in range(24)])
    mean, sem = runs.mean(axis=0), runs.std(axis=0, ddof=1) / math.sqrt(runs.shape[0])
    big = np.abs(q_exp) > 1e-3 * np.abs(q_exp).max()
    assert big.sum() >= 2
    assert np.all(np.abs(mean - q_exp)[big] <= 5 * sem[big] + 1e-6 * np.abs(q_exp).max())
    assert np.all(sem[big] > 0)                                   # the draws do differ from seed to seed


# ------------------------------------------------------------------ O7 truth association (reading D26)

def _collect_lut(p):
    """Hand-made LUT: an electron above the centre pixel of the window is collected whole during its arrival tick
    (LUT tick K - 1), nothing is induced anywhere else."""
    nb, Wp, K = p["bins_per_pixel"], p["window_pixels"], p["lut_ticks"]
    lut = np.zeros((Wp * nb, Wp * nb, K), dtype=np.float32)
    h = (Wp - 1) // 2
    lut[h * nb:(h + 1) * nb, h * nb:(h + 1) * nb, K - 1] = 1.0
    return lut


def test_hit_truth_hand_case():
    """Four short segments at the anode (sigma = 0) above pixel (4, 4) and one above its neighbour, under a LUT that
    collects a charge whole at its arrival tick (readout tick j + K - 1, K = 8).  Arrival ticks 12, 20, 30, 60 ->
    readout ticks 19, 27, 37, 67.  Charges: s0 alone stays below 7000 e-, s0 + s1 crosses at tick 27, the sample comes at
    43 and holds s0 + s1 + s2 (s2 arrives during the hold, D15); s3 crosses alone at 67, sample 83, integrated from tick
    44 on.  Shares are the charges themselves, fractions their ratios; the neighbour's segment s4 feeds nothing."""
    p = W.default_params(lut_ticks=8, n_readout_ticks=120)
    tpcs = [W.make_tpc(0.0, 0.0, 0.0, +1, 5.0, 9, 9, 0)]
    lut = _collect_lut(p)
    pitch = p["pixel_pitch_cm"]
    x, y = 4.5 * pitch, 4.5 * pitch
    f = lambda v: np.asarray(v, dtype=np.float32)
    t = [1.23, 2.05, 3.04, 6.0, 2.05]
    xs = [x, x + 0.01, x - 0.02, x, x - pitch]
    dE = [0.15, 0.11, 0.05, 0.30, 0.4]
    # 1 mm pieces along x (N = 100 sample points, all above the pixel and in one arrival tick)
    seg = dict(xs=f([v - 0.05 for v in xs]), ys=f([y] * 5), zs=f([0.0] * 5), ts=f(t), xe=f([v + 0.05 for v in xs]), ye=f([y] * 5),
               ze=f([0.0] * 5), te=f(t), dE=f(dE))
    _, ne, dr, pm = _chain(p, tpcs, seg)
    q = dr["q_a"]
    assert np.all(dr["sigma_T"] == 0.0) and np.allclose(q, ne)
    assert q[0] < 7000 <= q[0] + q[1] and q[3] >= 7000 and q[2] > 500
    waves, _ = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [4], [4])
    hp, ht, ha, _ = oracle.electronics(p, 0, [40], waves)
    assert ht.tolist() == [27 + 16, 67 + 16]
    sw = oracle.segment_currents(p, tpcs, lut, dr, pm, 0, 4, 4, np.arange(5))
    assert sw.shape == (5, 120)
    for s, n in enumerate((19, 27, 37, 67)):                     # each segment alone: its charge at its readout tick
        want = np.zeros(120)
        want[n] = q[s]
        assert np.allclose(sw[s], want, rtol=1e-12, atol=0)
    assert not sw[4].any()
    n0, share = oracle.hit_truth(p, ht, sw)
    assert n0.tolist() == [0, 44]
    assert np.allclose(share[0], [q[0], q[1], q[2], 0.0, 0.0], rtol=1e-12)
    assert np.allclose(share[1], [0.0, 0.0, 0.0, q[3], 0.0], rtol=1e-12)
    frac = share / share.sum(axis=1, keepdims=True)
    assert frac[0, 0] == pytest.approx(q[0] / (q[0] + q[1] + q[2]), rel=1e-12) and frac[1, 3] == 1.0
    # the sampled charge is what the ADC digitised (no noise): shares add up to it
    assert ha.tolist() == [_adc(q[0] + q[1] + q[2]), _adc(q[3])]


def test_hit_truth_periodic_reset_window():
    """Window start with the periodic reset (D17 / D26): 1000 e-/tick from two segments (600 + 400), period 7.  The
    electronics pin above gives samples at 22, 50, 78, each holding 23 ticks of charge: hit 0 integrates ticks 0..22 (no
    reset at tick 0, the resets at 7, 14, 21 fall in its hold), hit 1 ticks 28..50 -- the reset at tick 28 clears what
    ticks 23..27 brought, and tick 28 itself is integrated --, hit 2 ticks 56..78."""
    p = W.default_params(n_readout_ticks=100, periodic_reset_ticks=7)
    sw = np.stack([np.full(100, 600.0), np.full(100, 400.0)])
    hp, ht, ha, _ = oracle.electronics(p, 0, [9], sw.sum(axis=0)[None, :])
    assert ht.tolist() == [22, 50, 78]
    n0, share = oracle.hit_truth(p, ht, sw)
    assert n0.tolist() == [0, 28, 56]
    assert np.array_equal(share, np.array([[13800.0, 9200.0]] * 3))
    # without the reset the window of a later hit starts right after the previous sample
    p2 = W.default_params(n_readout_ticks=100)
    ht2 = oracle.electronics(p2, 0, [9], sw.sum(axis=0)[None, :])[1]
    assert ht2.tolist() == [22, 45, 68, 91]
    n0, share = oracle.hit_truth(p2, ht2, sw)
    assert n0.tolist() == [0, 23, 46, 69] and np.array_equal(share[1], [600.0 * 23, 400.0 * 23])


def test_hit_truth_sums_to_the_sampled_charge():
    """A diffused track over several pixels, analytic pad LUT: for every hit the shares of all segments add up to the
    integral of the pixel's total waveform (orc_pixel_current on all segments at once, a different summation order)
    over the hit's window, that integral reproduces the noise-free ADC code, the fractions add up to one, and every
    segment's shares over all hits of a pixel plus what was never sampled add up to its integrated current."""
    p, tpcs, lut = _small_setup(nx=10, ny=10, drift=6.0)
    pitch = p["pixel_pitch_cm"]
    seg = W.line_segments([2.2 * pitch, 3.4 * pitch, 1.0], [7.6 * pitch, 5.1 * pitch, 3.0], 0.1, 0.0, W._mip(6.0))
    _, ne, dr, pm = _chain(p, tpcs, seg)
    n = len(dr["q_a"])
    checked = 0
    for ix, iy in [(3, 3), (4, 4), (5, 4), (6, 4), (7, 5)]:
        waves, _ = oracle.pixel_currents(p, tpcs, lut, dr, pm, 0, [ix], [iy])
        hp, ht, ha, _ = oracle.electronics(p, 0, [iy * 10 + ix], waves)
        if len(ht) == 0:
            continue
        sw = oracle.segment_currents(p, tpcs, lut, dr, pm, 0, ix, iy, np.arange(n))
        assert np.allclose(sw.sum(axis=0), waves[0], rtol=1e-9, atol=1e-9 * np.abs(waves[0]).max())
        n0, share = oracle.hit_truth(p, ht, sw)
        for h in range(len(ht)):
            want = waves[0][n0[h]:ht[h] + 1].sum()
            assert share[h].sum() == pytest.approx(want, rel=1e-9)
            assert ha[h] == _adc(want)
            assert (share[h] / share[h].sum()).sum() == pytest.approx(1.0, abs=1e-12)
            assert n0[h] == (0 if h == 0 else ht[h - 1] + 1)
        rest = sw[:, ht[-1] + 1:].sum(axis=1)
        assert np.allclose(share.sum(axis=0) + rest, sw.sum(axis=1), rtol=1e-9, atol=1e-6)
        checked += len(ht)
    assert checked >= 4
