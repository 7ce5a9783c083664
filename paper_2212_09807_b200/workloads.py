"""Seeded synthetic inputs for the LArTPC charge hot path (arXiv 2212.09807).

This module is the ONE piece shared by the CUDA path (``lartpc``), the CPU
oracle (``oracle/``), the tests and ``bench.py``.  It holds inputs only:

* the parameter dictionary (constants the paper quotes, eqs. 3.1/3.2,
  P:L614 eq. 3.5, section 3.4; everything else per SURVEY.md 8(b)),
* TPC geometry tables for the five BASELINE.json configs,
* energy-deposit segment generators shaped like the paper's workloads
  (eq. 2.1: ``S_i = (r_s, r_e, E)_i``), standing in for the
  CORSIKA / edep-sim samples of P:L836 which are not available here,
* the harness response look-up table: the analytic weighting potential of a
  square pad differenced along a straight drift path (Shockley-Ramo, eq. 3.6
  P:L622-626; construction in SURVEY.md 8(c.2)).  It is an INPUT of
  ``lartpc_sim_create`` / of the oracle, not part of the method.

None of the method's arithmetic (recombination, drift, diffusion weights,
current sums, electronics) lives here; neither side imports the other.
All randomness comes from ``numpy.random.Generator(PCG64(seed))``.
"""
from __future__ import annotations

import dataclasses
import hashlib
import math
from typing import Dict, List, Optional

import numpy as np

PITCH_CM = 0.4434            # 0.4434 x 0.4434 cm^2 pads (31.038 cm / 70)
SEED_BASE = 0x22120980       # seed of config k = SEED_BASE + k

SEG_FIELDS = ("xs", "ys", "zs", "ts", "xe", "ye", "ze", "te", "dE")


def default_params(**over) -> Dict[str, float]:
    """Parameter dictionary; field names follow ``lartpc_params_t`` (include/lartpc.h)."""
    p = dict(
        e_field_kv_cm=0.5, lar_density_g_cm3=1.38, w_ion_mev=23.6e-6,
        recomb_model=1,                       # 0 = Birks (eq. 3.1), 1 = modified Box (eq. 3.2)
        birks_ab=0.800, birks_kb=0.0486,
        box_alpha=0.93, box_beta=0.212,       # P:L583 gives 0.207; BASELINE configs[0] 0.212 (D7)
        v_drift_cm_us=0.16, lifetime_us=2200.0,
        d_long_cm2_us=4.0e-6, d_tran_cm2_us=8.8e-6,   # 4.0 and 8.8 cm^2/s
        tick_us=0.1, t_origin_us=0.0,
        pixel_pitch_cm=PITCH_CM, bins_per_pixel=10, window_pixels=5, lut_ticks=200,
        n_readout_ticks=825,
        sample_step_cm=1.0e-3, n_sigma_map=5.0,       # 10 um sampling
        gain_mv_per_ke=4.0, v_cm_mv=288.0, v_ref_mv=1300.0, v_pedestal_mv=580.0, adc_bits=8,
        threshold_e=7000.0, hold_ticks=16, min_spacing_ticks=11, periodic_reset_ticks=0,
        noise_reset_e=0.0, noise_disc_e=0.0, noise_uncorr_e=0.0,
        max_hits_per_pixel=32,
    )
    for k, v in over.items():
        if k not in p:
            raise KeyError(k)
        p[k] = v
    return p


def make_tpc(x0, y0, z_anode, drift_sign, drift_len, nx, ny, first_pixel_id):
    return dict(x0=float(x0), y0=float(y0), z_anode=float(z_anode), drift_sign=int(drift_sign),
                drift_len=float(drift_len), nx=int(nx), ny=int(ny), first_pixel_id=int(first_pixel_id))


@dataclasses.dataclass
class Workload:
    name: str
    seed: int
    params: Dict[str, float]
    tpcs: List[dict]
    segments: Dict[str, np.ndarray]       # nine float32 arrays (SEG_FIELDS), same length
    lut: np.ndarray                       # float32 [W*nb][W*nb][K], tick fastest
    disabled_pixels: Optional[np.ndarray] = None   # sorted int32 global pixel ids (c2: 7.8 %)
    notes: str = ""

    @property
    def n_segments(self) -> int:
        return int(self.segments["xs"].shape[0])

    @property
    def n_pixels(self) -> int:
        return int(sum(t["nx"] * t["ny"] for t in self.tpcs))

    def sha256(self) -> Dict[str, str]:
        return {k: hashlib.sha256(np.ascontiguousarray(self.segments[k]).tobytes()).hexdigest()
                for k in SEG_FIELDS}

    def subset(self, idx) -> "Workload":
        seg = {k: np.ascontiguousarray(v[idx]) for k, v in self.segments.items()}
        return dataclasses.replace(self, segments=seg)


# --------------------------------------------------------------------------------------
# Response LUT of an ideal square pad; Shockley-Ramo eq. (3.6)
# --------------------------------------------------------------------------------------

def pad_weighting_potential(x, y, z, half_width):
    """W(x,y,z) of a square pad of half-width a on an infinite grounded plane, z > 0."""
    a = half_width

    def f(s, t):
        return np.arctan(s * t / (z * np.sqrt(s * s + t * t + z * z)))

    return (f(x + a, y + a) - f(x + a, y - a) - f(x - a, y + a) + f(x - a, y - a)) / (2.0 * math.pi)


def pad_response_lut(params) -> np.ndarray:
    """R[cy][cx][k]: electrons induced during LUT tick k by one electron that drifts
    straight down at v_d over bin (cx, cy) of the W x W pixel window and lands at the
    end of tick K-1.  Each series sums to exactly 1 (bins over the centre pixel) or 0."""
    nb, W, K = int(params["bins_per_pixel"]), int(params["window_pixels"]), int(params["lut_ticks"])
    pitch, dt, vd = params["pixel_pitch_cm"], params["tick_us"], params["v_drift_cm_us"]
    nbin = W * nb
    binw = pitch / nb
    c = (np.arange(nbin) + 0.5) * binw - 0.5 * W * pitch          # bin centres about the centre pixel
    X, Y = np.meshgrid(c, c, indexing="xy")                          # [cy][cx]
    inside = ((np.abs(X) < 0.5 * pitch) & (np.abs(Y) < 0.5 * pitch)).astype(np.float64)
    # potential at the START of tick k: height (K-k) * dt * vd, k = 1..K-1 ; at k = K the pad itself.
    wz = np.empty((K + 1, nbin, nbin), dtype=np.float64)
    wz[0] = 0.0                                                       # z = infinity (tick 0 absorbs the tail)
    for k in range(1, K):
        wz[k] = pad_weighting_potential(X, Y, (K - k) * dt * vd, 0.5 * pitch)
    wz[K] = inside                                                    # W(x, y, 0+)
    R = np.diff(wz, axis=0)                                           # [K][cy][cx]
    return np.ascontiguousarray(np.transpose(R, (1, 2, 0)).astype(np.float32))


# --------------------------------------------------------------------------------------
# Segment building blocks
# --------------------------------------------------------------------------------------

def _empty_segments():
    return {k: np.zeros(0, dtype=np.float32) for k in SEG_FIELDS}


def _concat(parts):
    if not parts:
        return _empty_segments()
    return {k: np.concatenate([p[k] for p in parts]).astype(np.float32) for k in SEG_FIELDS}


def line_segments(p0, p1, step_cm, t0, dedx_fn):
    """Cut the straight line p0->p1 into pieces of ``step_cm`` (last one shorter).
    ``dedx_fn(s_mid, length_total, n)`` returns dE/dx [MeV/cm] per piece."""
    p0 = np.asarray(p0, dtype=np.float64)
    p1 = np.asarray(p1, dtype=np.float64)
    length = float(np.linalg.norm(p1 - p0))
    if length <= 0.0:
        return _empty_segments()
    n = max(1, int(math.ceil(length / step_cm - 1e-9)))
    edges = np.minimum(np.arange(n + 1) * step_cm, length)
    d = (p1 - p0) / length
    s = p0[None, :] + edges[:-1, None] * d[None, :]
    e = p0[None, :] + edges[1:, None] * d[None, :]
    seg_len = edges[1:] - edges[:-1]
    dedx = np.asarray(dedx_fn(0.5 * (edges[1:] + edges[:-1]), length, n), dtype=np.float64)
    out = dict(xs=s[:, 0], ys=s[:, 1], zs=s[:, 2], ts=np.full(n, t0),
               xe=e[:, 0], ye=e[:, 1], ze=e[:, 2], te=np.full(n, t0), dE=dedx * seg_len)
    return {k: v.astype(np.float32) for k, v in out.items()}


def _volume_bounds(tpcs, pitch):
    """Axis-aligned box of each TPC drift volume: (xlo, xhi, ylo, yhi, zlo, zhi)."""
    b = []
    for t in tpcs:
        zlo, zhi = sorted((t["z_anode"], t["z_anode"] + t["drift_sign"] * t["drift_len"]))
        b.append((t["x0"], t["x0"] + t["nx"] * pitch, t["y0"], t["y0"] + t["ny"] * pitch, zlo, zhi))
    return np.asarray(b, dtype=np.float64)


def keep_inside(seg, tpcs, pitch):
    """Drop pieces whose midpoint lies in no TPC volume (tracks clipped at TPC boundaries, D8)."""
    if seg["xs"].shape[0] == 0:
        return seg
    b = _volume_bounds(tpcs, pitch)
    xm = 0.5 * (seg["xs"].astype(np.float64) + seg["xe"])
    ym = 0.5 * (seg["ys"].astype(np.float64) + seg["ye"])
    zm = 0.5 * (seg["zs"].astype(np.float64) + seg["ze"])
    inside = np.zeros(xm.shape[0], dtype=bool)
    margin = 1e-4
    for (xlo, xhi, ylo, yhi, zlo, zhi) in b:
        inside |= ((xm > xlo + margin) & (xm < xhi - margin) & (ym > ylo + margin) & (ym < yhi - margin)
                   & (zm > zlo + margin) & (zm < zhi - margin))
    return {k: v[inside] for k, v in seg.items()}


def _iso_dir(rng, n=None):
    cz = rng.uniform(-1.0, 1.0, size=n)
    ph = rng.uniform(0.0, 2.0 * math.pi, size=n)
    st = np.sqrt(1.0 - cz * cz)
    return np.stack([st * np.cos(ph), st * np.sin(ph), cz], axis=-1)


def _mip(dedx):
    return lambda s, L, n: np.full(n, dedx)


def _bragg(s, L, n):
    """Proton-like ramp: dE/dx ~ residual range^-0.42, about 5 MeV/cm far from the end, 30 at the end."""
    resid = np.maximum(L - s, 1e-3)
    return np.clip(30.0 * (resid / 0.4) ** -0.42, 5.0, 30.0)


def shower_segments(rng, vertex, axis, n_seg, t0, seg_len=0.05, x0_cm=14.0, r_cm=2.0, mean_de=0.1):
    """EM-shower-like cloud: n_seg pieces of 0.5 mm scattered about ``axis``; depth ~ Gamma(3, X0/2),
    radius ~ Exp(r_cm), energies ~ Exp(mean 0.1 MeV)."""
    axis = np.asarray(axis, dtype=np.float64)
    axis = axis / np.linalg.norm(axis)
    ref = np.array([1.0, 0.0, 0.0]) if abs(axis[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
    e1 = np.cross(axis, ref)
    e1 /= np.linalg.norm(e1)
    e2 = np.cross(axis, e1)
    depth = rng.gamma(3.0, x0_cm / 2.0, size=n_seg)
    rad = rng.exponential(r_cm, size=n_seg)
    ph = rng.uniform(0.0, 2.0 * math.pi, size=n_seg)
    mid = (np.asarray(vertex)[None, :] + depth[:, None] * axis[None, :]
           + (rad * np.cos(ph))[:, None] * e1[None, :] + (rad * np.sin(ph))[:, None] * e2[None, :])
    d = _iso_dir(rng, n_seg)
    s = mid - 0.5 * seg_len * d
    e = mid + 0.5 * seg_len * d
    de = rng.exponential(mean_de, size=n_seg)
    out = dict(xs=s[:, 0], ys=s[:, 1], zs=s[:, 2], ts=np.full(n_seg, t0),
               xe=e[:, 0], ye=e[:, 1], ze=e[:, 2], te=np.full(n_seg, t0), dE=de)
    return {k: v.astype(np.float32) for k, v in out.items()}


def interaction(rng_trk, rng_sh, vertex, t0, n_shower_seg, forward=None):
    """One neutrino-like vertex: 3-10 tracks (MIPs 10-100 cm at 2.1 MeV/cm, protons 2-30 cm with a
    Bragg-like ramp) and two EM showers sharing ``n_shower_seg`` pieces.
    Tracks and showers draw from separate generators so the tracks do not change when the
    shower multiplicity is rescaled."""
    parts = []
    ntrk = int(rng_trk.integers(3, 11))
    for _ in range(ntrk):
        d = _iso_dir(rng_trk)
        if forward is not None:
            d = d + 1.5 * np.asarray(forward)
            d /= np.linalg.norm(d)
        if rng_trk.uniform() < 0.6:
            L = rng_trk.uniform(10.0, 100.0)
            parts.append(line_segments(vertex, vertex + L * d, 0.1, t0, _mip(2.1)))
        else:
            L = rng_trk.uniform(2.0, 30.0)
            parts.append(line_segments(vertex, vertex + L * d, 0.1, t0, _bragg))
    for frac in (0.6, 0.4):
        ns = int(n_shower_seg * frac)
        d = _iso_dir(rng_sh)
        if forward is not None:
            d = d + 1.5 * np.asarray(forward)
        if ns > 0:
            parts.append(shower_segments(rng_sh, vertex, d, ns, t0))
    return _concat(parts)


def _n_ticks(params, drift_len, spill_us):
    """Readout window: (spill + max drift)/dt + K, plus the 5-sigma tail and the 1.6 us hold."""
    t_max = spill_us + drift_len / params["v_drift_cm_us"]
    sig_t = math.sqrt(2.0 * params["d_long_cm2_us"] * drift_len / params["v_drift_cm_us"]) / params["v_drift_cm_us"]
    return int(math.ceil((t_max + params["n_sigma_map"] * sig_t) / params["tick_us"])) + int(params["lut_ticks"]) + 24


# --------------------------------------------------------------------------------------
# The five BASELINE.json configs
# --------------------------------------------------------------------------------------

def config0(seed=None) -> Workload:
    """c0 'PR1 ref model': one straight MIP muon, 100 x 1 mm, 32x32 pixels, drift 0-10 cm, noise off."""
    seed = SEED_BASE + 0 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    p = default_params(recomb_model=1, box_beta=0.212)
    nx = ny = 32
    side, drift = nx * PITCH_CM, 10.0
    tpcs = [make_tpc(0.0, 0.0, 0.0, +1, drift, nx, ny, 0)]
    while True:
        start = np.array([rng.uniform(0, side), rng.uniform(0, side), rng.uniform(0, drift)])
        d = _iso_dir(rng)
        end = start + 10.0 * d
        if (0 < end[0] < side) and (0 < end[1] < side) and (0 < end[2] < drift):
            break
    seg = line_segments(start, end, 0.1, 0.0, _mip(2.1))
    p["n_readout_ticks"] = _n_ticks(p, drift, 0.0)
    return Workload("c0_pr1_single_muon", seed, p, tpcs, seg, pad_response_lut(p),
                    notes="one MIP track, 100 segments of 1 mm, dE=0.21 MeV each, ModBox, noise off")


def _moyal_dedx(rng, mpv=1.8, scale=0.18):
    def fn(s, L, n):
        z = rng.standard_normal(n)
        return np.clip(mpv + scale * (-np.log(np.maximum(z * z, 1e-300))), 0.2, 50.0)
    return fn


def config1(seed=None, n_muons=20) -> Workload:
    """c1 cosmic muons in one TPC: 70x70 pixels, 30 cm drift, 20 through-going muons, noise on."""
    seed = SEED_BASE + 1 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    p = default_params(recomb_model=1, box_beta=0.212, noise_reset_e=900.0, noise_uncorr_e=500.0)
    nx = ny = 70
    side, drift = nx * PITCH_CM, 30.0
    tpcs = [make_tpc(0.0, 0.0, 0.0, +1, drift, nx, ny, 0)]
    parts = []
    for _ in range(n_muons):
        # enter through the top face (y = side), direction uniform over the downward hemisphere
        start = np.array([rng.uniform(0, side), side, rng.uniform(0, drift)])
        d = _iso_dir(rng)
        d[1] = -abs(d[1]) - 1e-3
        d /= np.linalg.norm(d)
        end = start + 200.0 * d
        parts.append(keep_inside(line_segments(start, end, 0.1, 0.0, _moyal_dedx(rng)), tpcs, PITCH_CM))
    p["n_readout_ticks"] = _n_ticks(p, drift, 0.0)
    return Workload("c1_cosmics_one_tpc", seed, p, tpcs, _concat(parts), pad_response_lut(p),
                    notes="%d muons from the top face, 1 mm steps clipped to the box, Moyal dE/dx" % n_muons)


def _modules_2x2():
    tpcs, pid = [], 0
    nx, ny, drift, gap = 140, 280, 30.0, 2.0
    for my in range(2):
        for mx in range(2):
            x0 = mx * (nx * PITCH_CM + gap)
            y0 = my * (ny * PITCH_CM + gap)
            for sign in (+1, -1):
                tpcs.append(make_tpc(x0, y0, -sign * drift, sign, drift, nx, ny, pid))
                pid += nx * ny
    return tpcs


def _scaled_events(seed, tpcs, n_vertices, target, spill_us, forward, extra=None, tol=0.05):
    """Generate ``n_vertices`` interactions; the shower multiplicity is scaled until the total
    number of segments inside the TPC volumes is ``target`` +- tol."""
    b = _volume_bounds(tpcs, PITCH_CM)
    lo = np.array([b[:, 0].min(), b[:, 2].min(), b[:, 4].min()])
    hi = np.array([b[:, 1].max(), b[:, 3].max(), b[:, 5].max()])
    n_extra = extra["xs"].shape[0] if extra is not None else 0

    def build(n_sh):
        parts, n_in = ([extra] if extra is not None else []), []
        for v in range(n_vertices):
            rt = np.random.Generator(np.random.PCG64([seed, v, 0]))
            rs = np.random.Generator(np.random.PCG64([seed, v, 1]))
            vtx = lo + (hi - lo) * (0.15 + 0.7 * rt.uniform(size=3))
            t0 = rt.uniform(0.0, spill_us) if spill_us > 0 else 0.0
            parts.append(keep_inside(interaction(rt, rs, vtx, t0, n_sh, forward), tpcs, PITCH_CM))
        return _concat(parts)

    n_tracks = build(0)["xs"].shape[0]
    n_sh = max(1, (target - n_tracks) // max(n_vertices, 1))
    seg = None
    for _ in range(10):
        seg = build(n_sh)
        n = seg["xs"].shape[0]
        if abs(n - target) <= tol * target or n_sh <= 1 and n > target:
            break
        kept = max(n - n_tracks, 1)                       # shower pieces that fell inside a TPC
        n_sh = max(1, int(round(n_sh * max(target - n_tracks, 1) / kept)))
    return seg


def config2(seed=None, target=100_000) -> Workload:
    """c2 neutrino-like interactions in a 2x2-module volume: 8 TPCs of 140x280 pixels, Birks, noise on."""
    seed = SEED_BASE + 2 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    p = default_params(recomb_model=0, noise_reset_e=900.0, noise_uncorr_e=500.0)
    tpcs = _modules_2x2()
    seg = _scaled_events(seed, tpcs, 10, target, 0.0, forward=None)
    p["n_readout_ticks"] = _n_ticks(p, 30.0, 0.0)
    npix = sum(t["nx"] * t["ny"] for t in tpcs)
    disabled = np.sort(rng.choice(npix, size=int(round(0.078 * npix)), replace=False)).astype(np.int32)
    return Workload("c2_neutrino_2x2", seed, p, tpcs, seg, pad_response_lut(p), disabled_pixels=disabled,
                    notes="10 vertices, MIPs + Bragg protons + EM showers (0.5 mm), scaled to %d segments" % target)


def _modules_ndlar():
    tpcs, pid = [], 0
    nx, ny, drift, gap = 226, 677, 50.0, 2.0
    for jz in range(5):
        zc = jz * (2 * drift + gap)
        for ix in range(7):
            x0 = ix * (nx * PITCH_CM + gap)
            for sign in (+1, -1):
                tpcs.append(make_tpc(x0, 0.0, zc - sign * drift, sign, drift, nx, ny, pid))
                pid += nx * ny
    return tpcs


def config3(seed=None, target=5_000_000) -> Workload:
    """c3 full ND-LAr-scale spill: 70 TPCs of 226x677 pixels, 50 cm drift, 50 interactions + 20 rock muons."""
    seed = SEED_BASE + 3 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    p = default_params(recomb_model=0, noise_reset_e=900.0, noise_uncorr_e=500.0)
    tpcs = _modules_ndlar()
    b = _volume_bounds(tpcs, PITCH_CM)
    lo = np.array([b[:, 0].min(), b[:, 2].min(), b[:, 4].min()])
    hi = np.array([b[:, 1].max(), b[:, 3].max(), b[:, 5].max()])
    spill = 10.0
    rock = []
    for _ in range(20):                                   # through-going rock muons along +x
        start = np.array([lo[0], rng.uniform(lo[1], hi[1]), rng.uniform(lo[2], hi[2])])
        d = np.array([1.0, rng.normal(0, 0.08), rng.normal(0, 0.08)])
        d /= np.linalg.norm(d)
        rock.append(keep_inside(line_segments(start, start + (hi[0] - lo[0]) * 1.1 * d, 0.1,
                                              rng.uniform(0, spill), _mip(2.1)), tpcs, PITCH_CM))
    scale = target / 5_000_000.0
    n_vtx = max(1, int(round(50 * min(1.0, scale * 4)))) if scale < 0.25 else 50
    seg = _scaled_events(seed, tpcs, n_vtx, target, spill, forward=(1.0, 0.0, 0.0), extra=_concat(rock))
    p["n_readout_ticks"] = _n_ticks(p, 50.0, spill)
    return Workload("c3_ndlar_spill", seed, p, tpcs, seg, pad_response_lut(p),
                    notes="%d interactions + 20 rock muons over a 10 us spill, scaled to %d segments" % (n_vtx, target))


def config4(seed=None, n_segments=100_000, seg_len_cm=0.1, drift_cm=30.0, window_pixels=5,
            lut_ticks=200, placement="track") -> Workload:
    """c4 induced-current sweep point: one 226x677 plane; track-like or uniformly scattered placement."""
    seed = SEED_BASE + 4 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    p = default_params(recomb_model=0, window_pixels=window_pixels, lut_ticks=lut_ticks)
    nx, ny = 226, 677
    max_drift = 51.0                                  # the 50 cm sweep point sits inside the volume, not on the cathode
    tpcs = [make_tpc(0.0, 0.0, 0.0, +1, max_drift, nx, ny, 0)]
    W, H = nx * PITCH_CM, ny * PITCH_CM
    parts, n = [], 0
    if placement == "track":
        while n < n_segments:
            L = min(100.0, (n_segments - n) * seg_len_cm)
            # tracks nearly parallel to the plane at the requested drift distance (+- 2 cm slope)
            th = rng.uniform(0, 2 * math.pi)
            dz = rng.uniform(-0.02, 0.02) if drift_cm > 0 else 0.0
            d = np.array([math.cos(th), math.sin(th), dz])
            d /= np.linalg.norm(d)
            c = np.array([rng.uniform(0.3 * W, 0.7 * W), rng.uniform(0.2 * H, 0.8 * H), drift_cm])
            s = line_segments(c - 0.5 * L * d, c + 0.5 * L * d, seg_len_cm, 0.0, _mip(2.1))
            s = keep_inside(s, tpcs, PITCH_CM) if drift_cm > 0 else s
            parts.append(s)
            n += s["xs"].shape[0]
        seg = _concat(parts)
        seg = {k: v[:n_segments] for k, v in seg.items()}
    else:
        mid = np.stack([rng.uniform(2, W - 2, n_segments), rng.uniform(2, H - 2, n_segments),
                        np.full(n_segments, drift_cm)], axis=-1)
        d = _iso_dir(rng, n_segments)
        if drift_cm <= 0:
            d[:, 2] = 0.0
            d /= np.linalg.norm(d, axis=1, keepdims=True)
        s, e = mid - 0.5 * seg_len_cm * d, mid + 0.5 * seg_len_cm * d
        seg = dict(xs=s[:, 0], ys=s[:, 1], zs=s[:, 2], ts=np.zeros(n_segments),
                   xe=e[:, 0], ye=e[:, 1], ze=e[:, 2], te=np.zeros(n_segments),
                   dE=np.full(n_segments, 2.1 * seg_len_cm))
        seg = {k: v.astype(np.float32) for k, v in seg.items()}
    p["n_readout_ticks"] = _n_ticks(p, max_drift, 0.0)
    return Workload("c4_current_sweep", seed, p, tpcs, seg, pad_response_lut(p),
                    notes="n=%d len=%g cm drift=%g cm W=%d K=%d %s" % (n_segments, seg_len_cm, drift_cm,
                                                                       window_pixels, lut_ticks, placement))


def make_config(k: int, **kw) -> Workload:
    return (config0, config1, config2, config3, config4)[k](**kw)


# --------------------------------------------------------------------------------------
# Light simulation inputs: a synthetic stand-in for the Geant4-made light LUT of P:L744
# (visibility V_i[voxel] and relative arrival-time distribution f_i[voxel][time bin] per photosensor), sensor
# efficiencies and gains, a unit-normalised impulse response and a noise spectrum.  Inputs only, no method arithmetic.
# --------------------------------------------------------------------------------------
@dataclasses.dataclass
class LightSetup:
    params: Dict[str, float]
    eff: np.ndarray            # float32 [n_det] detection efficiency eps_i (eq. 4.2)
    gain: np.ndarray           # float32 [n_det] G_i of eq. (4.6), ADC per photoelectron
    vis: np.ndarray            # float32 [n_det][nvz][nvy][nvx] visibility V_i
    tprof: np.ndarray          # float32 [n_det][nvz][nvy][nvx][n_lut_t], sums to 1 over the last axis
    resp: np.ndarray           # float32 [n_resp] impulse response sampled at the tick, sums to 1
    noise_amp: np.ndarray      # float32 [n_noise] amplitudes of the noise sinusoids (ADC)
    noise_k: np.ndarray        # int32 [n_noise] their frequencies in cycles per waveform


def default_light_params(**over) -> Dict[str, float]:
    p = dict(w_ph_mev=19.5e-6, w_ion_mev=23.6e-6, tick_us=0.016, t_start_us=-0.32, n_ticks=1024, lut_m=2, n_lut_t=16,
             vox_x0=0.0, vox_y0=0.0, vox_z0=0.0, vox_size_cm=4.0, nvx=1, nvy=1, nvz=1, n_det=8,
             f_prompt=0.3, tau_prompt_us=0.007, tau_slow_us=1.6, trunc_tau=5.0, normal_above=30.0, n_resp=32, n_noise=0)
    p.update(over)
    return p


def light_setup(wl: "Workload", n_det: int = 16, vox_cm: float = 4.0, seed: Optional[int] = None, noise: bool = False,
                **over) -> LightSetup:
    """Voxel grid over the bounding box of the workload's TPCs, `n_det` sensors on the box's x faces, a solid-angle-like
    visibility that is exactly 0 beyond 1.5 m, arrival-time profiles that widen with distance."""
    rng = np.random.Generator(np.random.PCG64((wl.seed if seed is None else seed) + 77))
    pitch = wl.params["pixel_pitch_cm"]
    vb = _volume_bounds(wl.tpcs, pitch)
    x0, x1, y0, y1, z0, z1 = (float(vb[:, 0].min()), float(vb[:, 1].max()), float(vb[:, 2].min()), float(vb[:, 3].max()),
                              float(vb[:, 4].min()), float(vb[:, 5].max()))
    nv = [max(1, int(math.ceil((b - a) / vox_cm))) for a, b in ((x0, x1), (y0, y1), (z0, z1))]
    ts, te = wl.segments["ts"], wl.segments["te"]
    span = float(max(te.max(initial=0.0), ts.max(initial=0.0))) if len(ts) else 0.0
    p = default_light_params(vox_x0=x0, vox_y0=y0, vox_z0=z0, vox_size_cm=vox_cm, nvx=nv[0], nvy=nv[1], nvz=nv[2], n_det=n_det,
                             w_ion_mev=wl.params["w_ion_mev"], n_noise=24 if noise else 0)
    p.update(over)
    tail = p["trunc_tau"] * p["tau_slow_us"] + (p["n_lut_t"] * p["lut_m"] + p["n_resp"]) * p["tick_us"]
    if "n_ticks" not in over:
        p["n_ticks"] = int(math.ceil((span - p["t_start_us"] + tail) / p["tick_us"] / 64.0)) * 64
    # sensors on the two x faces of the box
    sx = np.where(np.arange(n_det) % 2 == 0, x0 - 1.0, x1 + 1.0)
    sy = rng.uniform(y0, y1, n_det)
    sz = rng.uniform(z0, z1, n_det)
    cx = x0 + (np.arange(nv[0]) + 0.5) * vox_cm
    cy = y0 + (np.arange(nv[1]) + 0.5) * vox_cm
    cz = z0 + (np.arange(nv[2]) + 0.5) * vox_cm
    Z, Y, X = np.meshgrid(cz, cy, cx, indexing="ij")
    vis = np.zeros((n_det,) + Z.shape, dtype=np.float32)
    tprof = np.zeros((n_det,) + Z.shape + (p["n_lut_t"],), dtype=np.float32)
    b = np.arange(p["n_lut_t"], dtype=np.float64)
    for i in range(n_det):
        r = np.sqrt((X - sx[i]) ** 2 + (Y - sy[i]) ** 2 + (Z - sz[i]) ** 2)
        v = 0.04 * 25.0 / (r * r + 25.0)
        v[r > 150.0] = 0.0
        vis[i] = v.astype(np.float32)
        mean = 0.5 + r / 40.0                                   # later and wider with distance (scattering)
        width = 0.6 + r / 60.0
        f = np.exp(-0.5 * ((b[None, None, None, :] - mean[..., None]) / width[..., None]) ** 2) + 1e-3
        tprof[i] = (f / f.sum(axis=-1, keepdims=True)).astype(np.float32)
    eff = rng.uniform(0.002, 0.006, n_det).astype(np.float32)
    gain = rng.uniform(8.0, 12.0, n_det).astype(np.float32)
    k = np.arange(p["n_resp"], dtype=np.float64)
    resp = (k + 0.5) * np.exp(-(k + 0.5) / 4.0)
    resp = (resp / resp.sum()).astype(np.float32)
    namp = (2.0 / (1.0 + np.arange(p["n_noise"]))).astype(np.float32)
    nk = (3 + 7 * np.arange(p["n_noise"])).astype(np.int32)
    return LightSetup(p, eff, gain, vis, tprof, resp, namp, nk)
