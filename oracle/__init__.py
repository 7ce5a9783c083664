"""ctypes front-end of the fp64 CPU oracle (``lartpc_oracle.c``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the CUDA product path never does and
shares nothing with it.  Every function cites the passage of arXiv 2212.09807 it follows in
``lartpc_oracle.c``.  Arrays in, numpy fp64 / int32 arrays out.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lartpc_oracle.c")
_LIB = os.path.join(_HERE, "liblartpc_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (fp contraction off so integer decisions are IEEE-exact)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                               _SRC, "-lm", "-o", _LIB])
    return _LIB


class OrcParams(C.Structure):
    _fields_ = [
        ("e_field", C.c_double), ("rho", C.c_double), ("w_ion", C.c_double),
        ("recomb_model", C.c_int),
        ("birks_ab", C.c_double), ("birks_kb", C.c_double), ("box_alpha", C.c_double), ("box_beta", C.c_double),
        ("v_drift", C.c_double), ("lifetime", C.c_double), ("d_long", C.c_double), ("d_tran", C.c_double),
        ("dt", C.c_double), ("t_origin", C.c_double), ("pitch", C.c_double),
        ("nb", C.c_int), ("wpix", C.c_int), ("klut", C.c_int), ("n_ticks", C.c_int),
        ("sample_step", C.c_double), ("n_sigma_map", C.c_double),
        ("gain_mv_per_ke", C.c_double), ("v_cm", C.c_double), ("v_ref", C.c_double), ("v_ped", C.c_double),
        ("adc_bits", C.c_int),
        ("threshold_e", C.c_double), ("hold_ticks", C.c_int), ("min_spacing_ticks", C.c_int),
        ("periodic_reset_ticks", C.c_int),
        ("noise_reset_e", C.c_double), ("noise_disc_e", C.c_double), ("noise_uncorr_e", C.c_double),
        ("max_hits_per_pixel", C.c_int),
    ]


class OrcTpc(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("z_anode", C.c_double), ("drift_sign", C.c_int),
                ("drift_len", C.c_double), ("nx", C.c_int), ("ny", C.c_int), ("first_pixel_id", C.c_int)]


_PARAM_MAP = dict(
    e_field="e_field_kv_cm", rho="lar_density_g_cm3", w_ion="w_ion_mev", recomb_model="recomb_model",
    birks_ab="birks_ab", birks_kb="birks_kb", box_alpha="box_alpha", box_beta="box_beta",
    v_drift="v_drift_cm_us", lifetime="lifetime_us", d_long="d_long_cm2_us", d_tran="d_tran_cm2_us",
    dt="tick_us", t_origin="t_origin_us", pitch="pixel_pitch_cm", nb="bins_per_pixel",
    wpix="window_pixels", klut="lut_ticks", n_ticks="n_readout_ticks",
    sample_step="sample_step_cm", n_sigma_map="n_sigma_map", gain_mv_per_ke="gain_mv_per_ke",
    v_cm="v_cm_mv", v_ref="v_ref_mv", v_ped="v_pedestal_mv", adc_bits="adc_bits",
    threshold_e="threshold_e", hold_ticks="hold_ticks", min_spacing_ticks="min_spacing_ticks",
    periodic_reset_ticks="periodic_reset_ticks", noise_reset_e="noise_reset_e",
    noise_disc_e="noise_disc_e", noise_uncorr_e="noise_uncorr_e", max_hits_per_pixel="max_hits_per_pixel",
)


def _params(d: Dict) -> OrcParams:
    p = OrcParams()
    for f, k in _PARAM_MAP.items():
        setattr(p, f, d[k])
    return p


def _tpcs(tpcs: Sequence[dict]):
    arr = (OrcTpc * len(tpcs))()
    for i, t in enumerate(tpcs):
        arr[i] = OrcTpc(t["x0"], t["y0"], t["z_anode"], t["drift_sign"], t["drift_len"], t["nx"], t["ny"],
                        t["first_pixel_id"])
    return arr


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_pixel_current.restype = C.c_double
        _lib.orc_electronics.restype = C.c_int
    return _lib


def set_threads(n: int) -> int:
    """Threads the per-pixel loops use from now on (OpenMP); returns the count in effect."""
    return int(_load().orc_set_threads(C.c_int(int(n))))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


def _fp(a):
    return _p(a, C.c_float)


def _dp(a):
    return _p(a, C.c_double)


def _ip(a):
    return _p(a, C.c_int32)


def quench(params, seg):
    """O1, eqs. (3.1)/(3.2): returns (dEdx [MeV/cm], n_e [electrons]) as fp64."""
    lib, n = _load(), seg["xs"].shape[0]
    s = {k: _f32(v) for k, v in seg.items()}
    dedx, ne = np.zeros(n), np.zeros(n)
    pp = _params(params)
    lib.orc_quench(C.byref(pp), C.c_int64(n), _fp(s["xs"]), _fp(s["ys"]), _fp(s["zs"]),
                   _fp(s["xe"]), _fp(s["ye"]), _fp(s["ze"]), _fp(s["dE"]), _dp(dedx), _dp(ne))
    return dedx, ne


def drift(params, tpcs, seg, n_e):
    """O2, eqs. (3.3)-(3.5): dict of per-segment drift quantities (fp64, tpc int32)."""
    lib, n = _load(), seg["xs"].shape[0]
    s = {k: _f32(v) for k, v in seg.items()}
    out = {k: np.zeros(n) for k in ("q_a", "sigma_T", "sigma_t", "u_s", "v_s", "u_e", "v_e", "T_s", "T_e")}
    out["tpc"] = np.zeros(n, dtype=np.int32)
    pp, tt = _params(params), _tpcs(tpcs)
    ne = np.ascontiguousarray(n_e, dtype=np.float64)
    lib.orc_drift(C.byref(pp), tt, C.c_int(len(tpcs)), C.c_int64(n),
                  _fp(s["xs"]), _fp(s["ys"]), _fp(s["zs"]), _fp(s["ts"]),
                  _fp(s["xe"]), _fp(s["ye"]), _fp(s["ze"]), _fp(s["te"]), _dp(ne),
                  _ip(out["tpc"]), _dp(out["q_a"]), _dp(out["sigma_T"]), _dp(out["sigma_t"]),
                  _dp(out["u_s"]), _dp(out["v_s"]), _dp(out["u_e"]), _dp(out["v_e"]),
                  _dp(out["T_s"]), _dp(out["T_e"]))
    return out


_PIX_KEYS = ("a_lo", "a_hi", "b_lo", "b_hi", "ix0", "ix1", "iy0", "iy1", "jt0", "jt1", "npix", "n_samples")


def pixmap(params, tpcs, seg, dr):
    """O3 (D10): dict of int32 arrays -- charged-bin box, pixel rectangle, arrival-tick range, npix, N."""
    lib, n = _load(), seg["xs"].shape[0]
    s = {k: _f32(v) for k, v in seg.items()}
    out = {k: np.zeros(n, dtype=np.int32) for k in _PIX_KEYS}
    pp, tt = _params(params), _tpcs(tpcs)
    lib.orc_pixmap(C.byref(pp), tt, C.c_int64(n),
                   _fp(s["xs"]), _fp(s["ys"]), _fp(s["zs"]), _fp(s["xe"]), _fp(s["ye"]), _fp(s["ze"]),
                   _ip(dr["tpc"]), _dp(dr["q_a"]), _dp(dr["sigma_T"]), _dp(dr["sigma_t"]),
                   _dp(dr["u_s"]), _dp(dr["v_s"]), _dp(dr["u_e"]), _dp(dr["v_e"]), _dp(dr["T_s"]), _dp(dr["T_e"]),
                   *[_ip(out[k]) for k in _PIX_KEYS])
    out["offsets"] = np.concatenate([[0], np.cumsum(out["npix"].astype(np.int64))])
    return out


def _seg_args(dr, pm):
    return (_ip(dr["tpc"]), _dp(dr["q_a"]), _dp(dr["sigma_T"]), _dp(dr["sigma_t"]),
            _dp(dr["u_s"]), _dp(dr["v_s"]), _dp(dr["u_e"]), _dp(dr["v_e"]), _dp(dr["T_s"]), _dp(dr["T_e"]),
            _ip(pm["n_samples"]))


def pixel_currents(params, tpcs, lut, dr, pm, tpc_index: int, ixs, iys, threads: Optional[int] = None):
    """O4+O5, eqs. (3.7)-(3.9): waveforms [len(ixs)][n_readout_ticks] (electrons per tick) and Q_p."""
    lib = _load()
    if threads is not None:
        lib.orc_set_threads(C.c_int(int(threads)))
    ixs = np.ascontiguousarray(ixs, dtype=np.int32)
    iys = np.ascontiguousarray(iys, dtype=np.int32)
    npx, nt = ixs.shape[0], int(params["n_readout_ticks"])
    waves, qp = np.zeros((npx, nt)), np.zeros(npx)
    lutc = _f32(lut)
    pp, tt = _params(params), _tpcs(tpcs)
    n = dr["tpc"].shape[0]
    lib.orc_plane_currents(C.byref(pp), tt, C.c_int(tpc_index), _fp(lutc), C.c_int64(n), *_seg_args(dr, pm),
                           C.c_int64(npx), _ip(ixs), _ip(iys), _dp(waves), _dp(qp))
    return waves, qp


def pixel_currents_random(params, tpcs, lut, dr, pm, tpc_index: int, ixs, iys, m_perturb: int, seed: int,
                          threads: Optional[int] = None):
    """O4r, eq. (3.9) as printed: M = ``m_perturb`` random perturbations per sample point (Philox-keyed by
    (seed; segment index, mu, nu)).  Returns waveforms [len(ixs)][n_readout_ticks] and Q_p."""
    lib = _load()
    if threads is not None:
        lib.orc_set_threads(C.c_int(int(threads)))
    ixs = np.ascontiguousarray(ixs, dtype=np.int32)
    iys = np.ascontiguousarray(iys, dtype=np.int32)
    npx, nt = ixs.shape[0], int(params["n_readout_ticks"])
    waves, qp = np.zeros((npx, nt)), np.zeros(npx)
    lutc = _f32(lut)
    pp = _params(params)
    n = dr["tpc"].shape[0]
    lib.orc_plane_currents_random(C.byref(pp), C.c_int(tpc_index), _fp(lutc), C.c_int64(n), *_seg_args(dr, pm),
                                  C.c_int(int(m_perturb)), C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF),
                                  C.c_int64(npx), _ip(ixs), _ip(iys), _dp(waves), _dp(qp))
    return waves, qp


def perturbation_normals(seed: int, s: int, mu: int, nu: int, clamp: float):
    """The three standard normals of perturbed point (segment s, mu, nu) (reading D25)."""
    lib = _load()
    z = (C.c_double * 3)()
    lib.orc_perturbation_normals(C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF), C.c_uint32(s), C.c_uint32(mu), C.c_uint32(nu),
                                 C.c_double(clamp), z)
    return np.array(list(z))


def direct_current(params, lut, dr, pm, tpc_index: int, ix: int, iy: int):
    """The literal nested sum of SURVEY.md 8(c.1) for one pixel (tiny inputs only)."""
    lib = _load()
    wave = np.zeros(int(params["n_readout_ticks"]))
    lutc = _f32(lut)
    pp = _params(params)
    n = dr["tpc"].shape[0]
    lib.orc_direct_current(C.byref(pp), C.c_int(tpc_index), _fp(lutc), C.c_int64(n), *_seg_args(dr, pm),
                           C.c_int(ix), C.c_int(iy), _dp(wave))
    return wave


def philox4x32_10(counter, key):
    lib = _load()
    c = (C.c_uint32 * 4)(*counter)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib.orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def noise_normals(seed: int, pixel_id: int, tick: int):
    lib = _load()
    z = (C.c_double * 3)()
    lib.orc_noise_normals(C.c_uint64(seed), C.c_uint32(pixel_id), C.c_uint32(tick), z)
    return [float(x) for x in z]


def electronics(params, seed: int, pixel_ids, waves, max_hits: Optional[int] = None):
    """O6 on each listed pixel: returns (hit_pixel, hit_tick, hit_adc) sorted by (pixel order given, tick),
    and hits-per-pixel counts (all hits counted even beyond ``max_hits``)."""
    lib = _load()
    pp = _params(params)
    mh = int(max_hits if max_hits is not None else params["max_hits_per_pixel"])
    waves = np.ascontiguousarray(waves, dtype=np.float64)
    hp, ht, ha, counts = [], [], [], []
    tick = np.zeros(mh, dtype=np.int32)
    adc = np.zeros(mh, dtype=np.int32)
    for i, pid in enumerate(np.asarray(pixel_ids).tolist()):
        nh = lib.orc_electronics(C.byref(pp), C.c_uint64(seed), C.c_int32(pid), _dp(waves[i]),
                                 C.c_int(mh), _ip(tick), _ip(adc))
        counts.append(nh)
        m = min(nh, mh)
        hp.extend([pid] * m)
        ht.extend(tick[:m].tolist())
        ha.extend(adc[:m].tolist())
    return (np.asarray(hp, dtype=np.int32), np.asarray(ht, dtype=np.int32), np.asarray(ha, dtype=np.int32),
            np.asarray(counts, dtype=np.int32))


def segment_currents(params, tpcs, lut, dr, pm, tpc_index: int, ix: int, iy: int, sel, threads: Optional[int] = None):
    """O7: I_{p,s}, eq. (3.9) for each listed segment alone, on pixel (ix, iy): [len(sel)][n_readout_ticks]."""
    lib = _load()
    if threads is not None:
        lib.orc_set_threads(C.c_int(int(threads)))
    sel = np.ascontiguousarray(sel, dtype=np.int64)
    nt = int(params["n_readout_ticks"])
    waves = np.zeros((len(sel), nt))
    lutc = _f32(lut)
    pp, tt = _params(params), _tpcs(tpcs)
    lib.orc_segment_currents(C.byref(pp), tt, C.c_int(tpc_index), _fp(lutc), *_seg_args(dr, pm),
                             C.c_int(int(ix)), C.c_int(int(iy)), C.c_int64(len(sel)), _p(sel, C.c_int64), _dp(waves))
    return waves


def hit_truth(params, hit_ticks, seg_waves):
    """O7 (reading D26): for the hits of ONE pixel (sample ticks in increasing order) and the per-segment currents
    ``seg_waves`` [n_sel][n_readout_ticks]: returns (n0 [n_hits] first integrated tick, share [n_hits][n_sel] electrons)."""
    lib = _load()
    pp = _params(params)
    ticks = np.ascontiguousarray(hit_ticks, dtype=np.int32)
    w = np.ascontiguousarray(seg_waves, dtype=np.float64)
    n0 = np.zeros(len(ticks), dtype=np.int32)
    share = np.zeros((len(ticks), w.shape[0]))
    lib.orc_hit_truth(C.byref(pp), C.c_int(len(ticks)), _ip(ticks), C.c_int64(w.shape[0]), _dp(w), _ip(n0), _dp(share))
    return n0, share


def active_pixels(tpcs, pm, dr, tpc_index: int):
    """Union of the O3 rectangles of one TPC: sorted (iy, ix) pairs, row-major order."""
    t = tpcs[tpc_index]
    mask = np.zeros((t["ny"], t["nx"]), dtype=bool)
    sel = np.nonzero((dr["tpc"] == tpc_index) & (pm["npix"] > 0))[0]
    for s in sel:
        mask[pm["iy0"][s]:pm["iy1"][s] + 1, pm["ix0"][s]:pm["ix1"][s] + 1] = True
    iy, ix = np.nonzero(mask)
    return ix.astype(np.int32), iy.astype(np.int32)


def run_chain(wl, pixels: Optional[Dict[int, tuple]] = None, threads: Optional[int] = None, seed: Optional[int] = None):
    """O1..O6 on a workload.  ``pixels`` optionally maps tpc index -> (ixs, iys) to restrict O4-O6 to a
    sample of pixels (used at sizes where the full plane would take hours).  Returns a dict."""
    dedx, ne = quench(wl.params, wl.segments)
    dr = drift(wl.params, wl.tpcs, wl.segments, ne)
    pm = pixmap(wl.params, wl.tpcs, wl.segments, dr)
    res = dict(dEdx=dedx, n_e=ne, drift=dr, pixmap=pm, pixel_id=[], waves=[], q_p=[])
    seed = wl.seed if seed is None else seed
    for ti, t in enumerate(wl.tpcs):
        if pixels is not None:
            if ti not in pixels:
                continue
            ixs, iys = pixels[ti]
        else:
            ixs, iys = active_pixels(wl.tpcs, pm, dr, ti)
        if len(ixs) == 0:
            continue
        waves, qp = pixel_currents(wl.params, wl.tpcs, wl.lut, dr, pm, ti, ixs, iys, threads)
        res["pixel_id"].append(t["first_pixel_id"] + np.asarray(iys, dtype=np.int64) * t["nx"] + np.asarray(ixs))
        res["waves"].append(waves)
        res["q_p"].append(qp)
    nt = int(wl.params["n_readout_ticks"])
    res["pixel_id"] = np.concatenate(res["pixel_id"]).astype(np.int32) if res["pixel_id"] else np.zeros(0, np.int32)
    res["waves"] = np.concatenate(res["waves"]) if res["waves"] else np.zeros((0, nt))
    res["q_p"] = np.concatenate(res["q_p"]) if res["q_p"] else np.zeros(0)
    hp, ht, ha, cnt = electronics(wl.params, seed, res["pixel_id"], res["waves"])
    res.update(hit_pixel=hp, hit_tick=ht, hit_adc=ha, hits_per_pixel=cnt)
    return res


# ---------------------------------------------------------------------------------------------------
# Light simulation: O8-O12 of lartpc_oracle.c
# ---------------------------------------------------------------------------------------------------
class OrcLightParams(C.Structure):
    _fields_ = [("w_ph", C.c_double), ("w_ion", C.c_double), ("dt", C.c_double), ("t_start", C.c_double),
                ("n_ticks", C.c_int), ("lut_m", C.c_int), ("n_lut_t", C.c_int),
                ("vx0", C.c_double), ("vy0", C.c_double), ("vz0", C.c_double), ("vsize", C.c_double),
                ("nvx", C.c_int), ("nvy", C.c_int), ("nvz", C.c_int), ("n_det", C.c_int),
                ("f_prompt", C.c_double), ("tau_p", C.c_double), ("tau_s", C.c_double), ("trunc_tau", C.c_double),
                ("normal_above", C.c_double), ("n_resp", C.c_int), ("n_noise", C.c_int)]


_LIGHT_MAP = dict(w_ph="w_ph_mev", w_ion="w_ion_mev", dt="tick_us", t_start="t_start_us", n_ticks="n_ticks", lut_m="lut_m",
                  n_lut_t="n_lut_t", vx0="vox_x0", vy0="vox_y0", vz0="vox_z0", vsize="vox_size_cm", nvx="nvx", nvy="nvy",
                  nvz="nvz", n_det="n_det", f_prompt="f_prompt", tau_p="tau_prompt_us", tau_s="tau_slow_us",
                  trunc_tau="trunc_tau", normal_above="normal_above", n_resp="n_resp", n_noise="n_noise")


def _light_params(d: Dict) -> OrcLightParams:
    p = OrcLightParams()
    for f, k in _LIGHT_MAP.items():
        setattr(p, f, d[k])
    return p


def light_npe(lp, seg, n_e, eff, vis):
    """O8, eqs. (4.1)(4.2): returns dict(vox int32[n], k0 int32[n], n_gamma[n], npe[n_det][n])."""
    lib, n = _load(), seg["xs"].shape[0]
    s = {k: _f32(v) for k, v in seg.items()}
    pp = _light_params(lp)
    nd = int(lp["n_det"])
    out = dict(vox=np.zeros(n, np.int32), k0=np.zeros(n, np.int32), n_gamma=np.zeros(n), npe=np.zeros((nd, n)))
    ne = np.ascontiguousarray(n_e, dtype=np.float64)
    lib.orc_light_npe(C.byref(pp), C.c_int64(n), _fp(s["xs"]), _fp(s["ys"]), _fp(s["zs"]), _fp(s["ts"]),
                      _fp(s["xe"]), _fp(s["ye"]), _fp(s["ze"]), _fp(s["te"]), _fp(s["dE"]), _dp(ne),
                      _fp(_f32(eff)), _fp(_f32(vis)), _ip(out["vox"]), _ip(out["k0"]), _dp(out["n_gamma"]), _dp(out["npe"]))
    return out


def light_profile(lp, vox, k0, npe, tprof):
    """O9, eq. (4.3): photoelectrons per tick [n_det][n_ticks]."""
    lib = _load()
    pp = _light_params(lp)
    ipe = np.zeros((int(lp["n_det"]), int(lp["n_ticks"])))
    lib.orc_light_profile(C.byref(pp), C.c_int64(len(vox)), _ip(np.ascontiguousarray(vox, np.int32)),
                          _ip(np.ascontiguousarray(k0, np.int32)), _dp(np.ascontiguousarray(npe, np.float64)),
                          _fp(_f32(tprof)), _dp(ipe))
    return ipe


def light_scint_weights(lp):
    """O10: the weights f_scint(s dt) dt of eq. (4.5), s = 0 .. floor(trunc_tau tau_s / dt)."""
    lib = _load()
    pp = _light_params(lp)
    cap = int(lp["trunc_tau"] * lp["tau_slow_us"] / lp["tick_us"]) + 8
    w = np.zeros(cap)
    s_max = lib.orc_light_scint_weights(C.byref(pp), _dp(w), C.c_int(cap))
    return w[:s_max + 1].copy()


def light_convolve(x, w, scale=None):
    """Truncated causal convolution of eq. (4.5) / the sum of eq. (4.6): x [n_det][n_ticks], w [n_w], scale [n_det] or None."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    out = np.zeros_like(x)
    sc = _fp(_f32(scale)) if scale is not None else None
    lib.orc_light_convolve(C.c_int(x.shape[0]), C.c_int(x.shape[1]), _dp(x), _dp(w), C.c_int(len(w)), sc, _dp(out))
    return out


def light_fluctuate(lp, seed: int, isc):
    """O11: observed photoelectrons per (sensor, tick) (Poisson below normal_above, normal at or above)."""
    lib = _load()
    pp = _light_params(lp)
    isc = np.ascontiguousarray(isc, dtype=np.float64)
    out = np.zeros_like(isc)
    lib.orc_light_fluctuate(C.byref(pp), C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF), _dp(isc), _dp(out))
    return out


def light_noise(lp, seed: int, amp, kf):
    """O12 noise term of eq. (4.6) (reading D33): [n_det][n_ticks]."""
    lib = _load()
    pp = _light_params(lp)
    out = np.zeros((int(lp["n_det"]), int(lp["n_ticks"])))
    lib.orc_light_noise(C.byref(pp), C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF), _fp(_f32(amp)),
                        _ip(np.ascontiguousarray(kf, np.int32)), _dp(out))
    return out


def light_chain(lp, ls, seg, n_e, seed: int):
    """O8-O12 in sequence on a workload's segments; `ls` carries eff, gain, vis, tprof, resp, noise_amp, noise_k."""
    a = light_npe(lp, seg, n_e, ls.eff, ls.vis)
    ipe = light_profile(lp, a["vox"], a["k0"], a["npe"], ls.tprof)
    isc = light_convolve(ipe, light_scint_weights(lp))
    nobs = light_fluctuate(lp, seed, isc)
    v = light_convolve(nobs, ls.resp.astype(np.float64), ls.gain)
    if int(lp["n_noise"]) > 0:
        v = v + light_noise(lp, seed, ls.noise_amp, ls.noise_k)
    return dict(a, ipe=ipe, isc=isc, nobs=nobs, v=v)
