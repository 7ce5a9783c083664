"""Thin Python binding of the C-ABI library ``liblartpc.so`` (include/lartpc.h).

Argument marshalling only: every step of the path runs in the library's sm_100a kernels.
PyTorch supplies device memory (``torch.empty(..., device="cuda")``) and the CUDA stream.
There is no CPU fallback: importing works anywhere, but creating a :class:`Sim` raises if the
library is missing or the device is not a compute-capability 10.x GPU.

Function names follow the C entry points: ``quench`` -> ``lartpc_quench`` (eqs. 3.1/3.2 of
arXiv 2212.09807), ``drift`` (eqs. 3.3-3.5), ``pixels_from_segments``,
``induced_current`` (eq. 3.9), ``sum_pixel_signals``, ``electronics``,
``run_spill``.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblartpc.so")
_lib = None

SEG_FIELDS = ("xs", "ys", "zs", "ts", "xe", "ye", "ze", "te", "dE")


class LartpcError(RuntimeError):
    pass


class Params(C.Structure):
    _fields_ = [
        ("e_field_kv_cm", C.c_double), ("lar_density_g_cm3", C.c_double), ("w_ion_mev", C.c_double),
        ("recomb_model", C.c_int),
        ("birks_ab", C.c_double), ("birks_kb", C.c_double), ("box_alpha", C.c_double), ("box_beta", C.c_double),
        ("v_drift_cm_us", C.c_double), ("lifetime_us", C.c_double),
        ("d_long_cm2_us", C.c_double), ("d_tran_cm2_us", C.c_double),
        ("tick_us", C.c_double), ("t_origin_us", C.c_double),
        ("pixel_pitch_cm", C.c_double),
        ("bins_per_pixel", C.c_int), ("window_pixels", C.c_int), ("lut_ticks", C.c_int),
        ("n_readout_ticks", C.c_int),
        ("sample_step_cm", C.c_double), ("n_sigma_map", C.c_double),
        ("gain_mv_per_ke", C.c_double), ("v_cm_mv", C.c_double), ("v_ref_mv", C.c_double),
        ("v_pedestal_mv", C.c_double),
        ("adc_bits", C.c_int),
        ("threshold_e", C.c_double),
        ("hold_ticks", C.c_int), ("min_spacing_ticks", C.c_int), ("periodic_reset_ticks", C.c_int),
        ("noise_reset_e", C.c_double), ("noise_disc_e", C.c_double), ("noise_uncorr_e", C.c_double),
        ("max_hits_per_pixel", C.c_int),
    ]


class Tpc(C.Structure):
    _fields_ = [("x0", C.c_double), ("y0", C.c_double), ("z_anode", C.c_double), ("drift_sign", C.c_int),
                ("drift_len", C.c_double), ("nx", C.c_int), ("ny", C.c_int), ("first_pixel_id", C.c_int)]


_P = C.c_void_p


class Segments(C.Structure):
    _fields_ = [(k, _P) for k in SEG_FIELDS]


class Drifted(C.Structure):
    _fields_ = [(k, _P) for k in ("tpc", "q_anode", "sigma_T", "sigma_t", "u_s", "v_s", "u_e", "v_e", "T_s", "T_e")]


_PIX_I32 = ("a_lo", "a_hi", "b_lo", "b_hi", "ix0", "ix1", "iy0", "iy1", "jt0", "jt1", "npix", "n_samples")


class Pixmap(C.Structure):
    _fields_ = [(k, _P) for k in _PIX_I32 + ("offsets",)]


class PixmapInfo(C.Structure):
    _fields_ = [("max_npix", C.c_int32), ("max_ticks", C.c_int32), ("total_npix", C.c_int64),
                ("n_active_segments", C.c_int64), ("n_tiles", C.c_int64), ("n_pairs", C.c_int64),
                ("n_active_pixels", C.c_int64), ("total_samples", C.c_int64),
                ("tile_targets", C.c_int32), ("tile_ticks", C.c_int32),
                ("tile_charge_floats", C.c_int32), ("tile_block", C.c_int32)]


class Signals(C.Structure):
    _fields_ = [("tile_capacity", C.c_int64), ("partial", _P), ("tile_range", _P), ("charge", _P)]


class Waveforms(C.Structure):
    _fields_ = [("pixel_capacity", C.c_int64), ("sample_capacity", C.c_int64), ("pixel_id", _P),
                ("first_tick", _P), ("length", _P), ("offset", _P), ("samples", _P),
                ("n_active", C.c_int64), ("total_samples", C.c_int64)]


class Hits(C.Structure):
    _fields_ = [("hit_capacity", C.c_int64), ("hit_pixel", _P), ("hit_tick", _P), ("hit_adc", _P),
                ("hits_per_pixel", _P), ("q_pixel", _P), ("counters", _P)]


class Truth(C.Structure):
    _fields_ = [("k_max", C.c_int32), ("reserved", C.c_int32), ("seg", _P), ("frac", _P), ("q_signal", _P), ("n_contrib", _P)]


class LightParams(C.Structure):
    _fields_ = [("w_ph_mev", C.c_double), ("w_ion_mev", C.c_double), ("tick_us", C.c_double), ("t_start_us", C.c_double),
                ("n_ticks", C.c_int), ("lut_m", C.c_int), ("n_lut_t", C.c_int),
                ("vox_x0", C.c_double), ("vox_y0", C.c_double), ("vox_z0", C.c_double), ("vox_size_cm", C.c_double),
                ("nvx", C.c_int), ("nvy", C.c_int), ("nvz", C.c_int), ("n_det", C.c_int),
                ("f_prompt", C.c_double), ("tau_prompt_us", C.c_double), ("tau_slow_us", C.c_double),
                ("trunc_tau", C.c_double), ("normal_above", C.c_double), ("n_resp", C.c_int), ("n_noise", C.c_int)]


class Stats(C.Structure):
    _fields_ = [(k, C.c_int64) for k in ("n_segments", "n_active_segments", "n_tiles", "n_pairs", "n_active_pixels",
                                        "total_samples", "n_hits", "n_hits_total", "n_pixels_overflow",
                                        "n_hits_dropped")] + \
               [("n_batches", C.c_int32), ("reserved", C.c_int32), ("flops_current", C.c_double)]


EXPORTS = ("lartpc_sim_create", "lartpc_sim_create_ex", "lartpc_response_mode", "lartpc_sim_destroy", "lartpc_set_disabled_pixels",
           "lartpc_set_random_perturbations", "lartpc_set_truncation_compensation", "lartpc_chunk_ticks",
           "lartpc_workspace_bytes", "lartpc_quench", "lartpc_drift", "lartpc_pixels_from_segments",
           "lartpc_induced_current", "lartpc_sum_pixel_signals", "lartpc_electronics", "lartpc_electronics_static", "lartpc_hit_truth",
           "lartpc_run_spill",
           "lartpc_readout_tiles", "lartpc_pack_hits",
           "lartpc_light_create", "lartpc_light_destroy", "lartpc_light_npe", "lartpc_light_profile",
           "lartpc_light_scintillation", "lartpc_light_fluctuate", "lartpc_light_electronics", "lartpc_light_workspace_bytes",
           "lartpc_light_run",
           "lartpc_measure_fp32_peak", "lartpc_set_profiling", "lartpc_get_stage_ms", "lartpc_get_counters", "lartpc_kernel_launches",
           "lartpc_strerror")


def load_library():
    """dlopen liblartpc.so; raises LartpcError when it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LartpcError("liblartpc.so is not built: run `python -m paper_2212_09807_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        lib = C.CDLL(LIB_PATH)
        lib.lartpc_strerror.restype = C.c_char_p
        lib.lartpc_workspace_bytes.restype = C.c_size_t
        lib.lartpc_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        lib.lartpc_kernel_launches.restype = C.c_int64
        lib.lartpc_sim_destroy.restype = None
        lib.lartpc_sim_destroy.argtypes = [C.c_void_p]
        lib.lartpc_light_destroy.restype = None
        lib.lartpc_light_destroy.argtypes = [C.c_void_p]
        lib.lartpc_light_workspace_bytes.restype = C.c_size_t
        lib.lartpc_light_workspace_bytes.argtypes = [C.c_void_p, C.c_int64]
        for name in EXPORTS:
            getattr(lib, name)
        _lib = lib
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        raise LartpcError("%s failed: %s (%d)" % (what, load_library().lartpc_strerror(rc).decode(), rc))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise LartpcError("no CUDA device: the LArTPC path runs only on an sm_100a GPU (no CPU fallback)")
    return torch


def _stream_ptr(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def measure_fp32_peak(variant: int = 0) -> float:
    """FP32 FMA rate in TFLOP/s from the library's FFMA-chain microbenchmark (0 scalar, 1 packed FFMA2)."""
    torch = _torch()
    out = C.c_double(0.0)
    _check(load_library().lartpc_measure_fp32_peak(C.c_int(variant), C.byref(out), _stream_ptr(torch)),
           "lartpc_measure_fp32_peak")
    return float(out.value)


def kernel_launches() -> int:
    """Kernels launched by the library in this process so far."""
    return int(load_library().lartpc_kernel_launches())


class Sim:
    """Owns a ``lartpc_sim_t`` (detector / physics parameters, TPC table, response LUT)."""

    RESPONSE_MODES = {"auto": 0, "tensor": 1, "ffma": 2}

    def __init__(self, params: Dict, tpcs: Sequence[dict], lut: np.ndarray, device: str = "cuda:0",
                 response: str = "auto"):
        """``response``: how S4 applies the LUT -- "tensor" (tcgen05), "ffma" (FP32 pipe) or "auto"."""
        torch = _torch()
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.lib = load_library()
        self.params = dict(params)
        self.tpcs = list(tpcs)
        p = Params()
        for name, _ in Params._fields_:
            setattr(p, name, params[name])
        arr = (Tpc * len(tpcs))()
        for i, t in enumerate(tpcs):
            arr[i] = Tpc(t["x0"], t["y0"], t["z_anode"], t["drift_sign"], t["drift_len"], t["nx"], t["ny"],
                         t["first_pixel_id"])
        lut = np.ascontiguousarray(lut, dtype=np.float32)
        h = C.c_void_p()
        _check(self.lib.lartpc_sim_create_ex(C.byref(p), arr, C.c_int(len(tpcs)),
                                             lut.ctypes.data_as(C.c_void_p), C.c_size_t(lut.size),
                                             C.c_int(self.RESPONSE_MODES[response]), C.byref(h)),
               "lartpc_sim_create_ex")
        self.handle = h
        self.response_mode = {1: "tensor", 2: "ffma"}[int(self.lib.lartpc_response_mode(self.handle))]
        self.chunk_ticks = int(self.lib.lartpc_chunk_ticks(self.handle))
        self.info: Optional[PixmapInfo] = None
        self._keep = {}

    def close(self):
        if getattr(self, "handle", None):
            self.lib.lartpc_sim_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers ------------------------------------------------------------------------------------
    def _empty(self, n, dtype):
        return self.torch.empty(int(max(n, 0)), dtype=dtype, device=self.device)

    def upload_segments(self, seg: Dict[str, np.ndarray]):
        """Host SoA arrays -> device tensors (one float32 tensor per field)."""
        t = self.torch
        return {k: t.from_numpy(np.ascontiguousarray(seg[k], dtype=np.float32)).to(self.device) for k in SEG_FIELDS}

    def _seg_struct(self, seg):
        s = Segments()
        n = None
        for k in SEG_FIELDS:
            v = seg[k]
            if v.dtype != self.torch.float32 or not v.is_cuda or not v.is_contiguous():
                raise LartpcError("segment field %s must be a contiguous float32 CUDA tensor" % k)
            n = v.numel() if n is None else n
            if v.numel() != n:
                raise LartpcError("segment fields differ in length")
            setattr(s, k, v.data_ptr())
        return s, int(n)

    def set_random_perturbations(self, m: int, seed: int = 0):
        """S4 as eq. (3.9) prints it: m random perturbations per sample point (0 = expectation form, the default)."""
        _check(self.lib.lartpc_set_random_perturbations(self.handle, C.c_int(int(m)),
                                                        C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF)),
               "lartpc_set_random_perturbations")

    def set_truncation_compensation(self, kappa: float):
        """Tensor-core response: expected relative truncation loss per accumulated product that the epilogue adds back
        (include/lartpc.h; 0 = off)."""
        _check(self.lib.lartpc_set_truncation_compensation(self.handle, C.c_double(float(kappa))),
               "lartpc_set_truncation_compensation")

    def set_disabled_pixels(self, ids: np.ndarray):
        ids = np.ascontiguousarray(ids, dtype=np.int32)
        _check(self.lib.lartpc_set_disabled_pixels(self.handle, ids.ctypes.data_as(C.c_void_p), C.c_int64(ids.size)),
               "lartpc_set_disabled_pixels")

    # -- stages -------------------------------------------------------------------------------------
    def quench(self, seg):
        """S1: returns (dEdx, n_e) float32 tensors."""
        t = self.torch
        s, n = self._seg_struct(seg)
        dedx, ne = self._empty(n, t.float32), self._empty(n, t.float32)
        _check(self.lib.lartpc_quench(self.handle, C.byref(s), C.c_int64(n), C.c_void_p(dedx.data_ptr()),
                                      C.c_void_p(ne.data_ptr()), _stream_ptr(t)), "lartpc_quench")
        return dedx, ne

    def drift(self, seg, n_e):
        """S2: returns a dict of tensors named like ``lartpc_drifted_t``."""
        t = self.torch
        s, n = self._seg_struct(seg)
        out = dict(tpc=self._empty(n, t.int32), q_anode=self._empty(n, t.float32),
                   sigma_T=self._empty(n, t.float32), sigma_t=self._empty(n, t.float32))
        for k in ("u_s", "v_s", "u_e", "v_e", "T_s", "T_e"):
            out[k] = self._empty(n, t.float64)
        d = Drifted(**{k: v.data_ptr() for k, v in out.items()})
        _check(self.lib.lartpc_drift(self.handle, C.byref(s), C.c_int64(n), C.c_void_p(n_e.data_ptr()), C.byref(d),
                                     _stream_ptr(t)), "lartpc_drift")
        out["_struct"] = d
        return out

    def pixels_from_segments(self, seg, drifted):
        """S3: returns (pixmap dict, PixmapInfo).  Synchronises the stream once (sizes go to the host)."""
        t = self.torch
        s, n = self._seg_struct(seg)
        out = {k: self._empty(n, t.int32) for k in _PIX_I32}
        out["offsets"] = self._empty(n + 1, t.int64)
        pm = Pixmap(**{k: v.data_ptr() for k, v in out.items()})
        info = PixmapInfo()
        _check(self.lib.lartpc_pixels_from_segments(self.handle, C.byref(s), C.byref(drifted["_struct"]),
                                                    C.c_int64(n), C.byref(pm), C.byref(info), _stream_ptr(t)),
               "lartpc_pixels_from_segments")
        out["_struct"] = pm
        out["_n"] = n
        self.info = info
        return out, info

    def induced_current(self, drifted, pixmap):
        """S4: returns the signals dict (tile partial waveforms)."""
        t = self.torch
        info = self.info
        nt = int(info.n_tiles)
        blk = max(int(info.tile_block), 1)               # the tensor-core operand image comes in whole units of tiles
        nt_cap = (nt + blk - 1) // blk * blk
        out = dict(partial=self._empty(nt * info.tile_targets * info.tile_ticks, t.float32),
                   tile_range=self._empty(nt * 4, t.int32),
                   charge=self._empty(nt_cap * info.tile_charge_floats, t.float32))
        sig = Signals(nt_cap, out["partial"].data_ptr(), out["tile_range"].data_ptr(), out["charge"].data_ptr())
        _check(self.lib.lartpc_induced_current(self.handle, C.byref(drifted["_struct"]), C.byref(pixmap["_struct"]),
                                               C.c_int64(pixmap["_n"]), C.byref(sig), _stream_ptr(t)),
               "lartpc_induced_current")
        out["_struct"] = sig
        return out

    def sum_pixel_signals(self, signals):
        """S5: returns the waveforms dict (pixel_id, first_tick, length, offset, samples)."""
        t = self.torch
        info = self.info
        na, ns = int(info.n_active_pixels), int(info.total_samples)
        out = dict(pixel_id=self._empty(na, t.int32), first_tick=self._empty(na, t.int32),
                   length=self._empty(na, t.int32), offset=self._empty(na + 1, t.int64),
                   samples=self._empty(ns, t.float32))
        wf = Waveforms(na, ns, out["pixel_id"].data_ptr(), out["first_tick"].data_ptr(), out["length"].data_ptr(),
                       out["offset"].data_ptr(), out["samples"].data_ptr(), 0, 0)
        _check(self.lib.lartpc_sum_pixel_signals(self.handle, C.byref(signals["_struct"]), C.byref(wf),
                                                 _stream_ptr(t)), "lartpc_sum_pixel_signals")
        out["_struct"] = wf
        return out

    def _hits(self, capacity, n_active):
        t = self.torch
        out = dict(hit_pixel=self._empty(capacity, t.int32), hit_tick=self._empty(capacity, t.int32),
                   hit_adc=self._empty(capacity, t.int32), counters=t.zeros(4, dtype=t.int64, device=self.device))
        if n_active is not None:
            out["hits_per_pixel"] = self._empty(n_active, t.int32)
            out["q_pixel"] = self._empty(n_active, t.float32)
        h = Hits(int(capacity), out["hit_pixel"].data_ptr(), out["hit_tick"].data_ptr(), out["hit_adc"].data_ptr(),
                 out["hits_per_pixel"].data_ptr() if n_active is not None else None,
                 out["q_pixel"].data_ptr() if n_active is not None else None, out["counters"].data_ptr())
        return out, h

    def electronics(self, waveforms, seed: int, hit_capacity: Optional[int] = None):
        """S6: returns the hits dict; ``counters`` = [written, total, pixels over capacity, dropped]."""
        t = self.torch
        na = int(waveforms["_struct"].n_active)
        cap = int(hit_capacity if hit_capacity is not None else na * self.params["max_hits_per_pixel"])
        out, h = self._hits(cap, na)
        _check(self.lib.lartpc_electronics(self.handle, C.byref(waveforms["_struct"]), C.c_uint64(seed), C.byref(h),
                                           _stream_ptr(t)), "lartpc_electronics")
        out["_struct"] = h
        return out

    def electronics_static(self, waveforms, seed: int, hit_capacity: Optional[int] = None):
        """S6 through lartpc_electronics_static: no allocation inside the library, scratch in a fixed device array
        (LARTPC_STATIC_MAX_PIXELS / LARTPC_STATIC_MAX_SLOTS: RuntimeError beyond them); same outputs as ``electronics``."""
        t = self.torch
        na = int(waveforms["_struct"].n_active)
        cap = int(hit_capacity if hit_capacity is not None else na * self.params["max_hits_per_pixel"])
        out, h = self._hits(cap, na)
        _check(self.lib.lartpc_electronics_static(self.handle, C.byref(waveforms["_struct"]), C.c_uint64(seed), C.byref(h),
                                                  _stream_ptr(t)), "lartpc_electronics_static")
        out["_struct"] = h
        return out

    def hit_truth(self, drifted, pixmap, hits, n_hits: Optional[int] = None, k_max: int = 4):
        """Truth association after the staged S6 (reading D26): per hit the ``k_max`` segments with the largest shares.
        Returns a dict: seg int32 [n_hits, k_max] (-1 = unused), frac float32 [n_hits, k_max], q_signal float32 [n_hits],
        n_contrib int32 [n_hits]."""
        t = self.torch
        n = int(hits["counters"][0].item()) if n_hits is None else int(n_hits)
        m = max(n, 1)
        out = dict(seg=self._empty(m * k_max, t.int32), frac=self._empty(m * k_max, t.float32),
                   q_signal=self._empty(m, t.float32), n_contrib=self._empty(m, t.int32))
        tr = Truth(k_max=int(k_max), reserved=0, **{k: v.data_ptr() for k, v in out.items()})
        n_seg = int(drifted["tpc"].numel())
        _check(self.lib.lartpc_hit_truth(self.handle, C.byref(drifted["_struct"]), C.byref(pixmap["_struct"]), C.c_int64(n_seg),
                                         C.byref(hits["_struct"]), C.c_int64(n), C.byref(tr), _stream_ptr(t)),
               "lartpc_hit_truth")
        return dict(seg=out["seg"][:n * k_max].view(n, k_max), frac=out["frac"][:n * k_max].view(n, k_max),
                    q_signal=out["q_signal"][:n], n_contrib=out["n_contrib"][:n])

    STAGES = ("quench", "drift", "pixels_from_segments", "induced_current_charge", "induced_current_response",
              "sum_pixel_signals", "electronics")

    def set_profiling(self, on: bool):
        _check(self.lib.lartpc_set_profiling(self.handle, C.c_int(1 if on else 0)), "lartpc_set_profiling")

    def stage_ms(self):
        """Per-stage device ms, launch counts and the S4 multiply-add count of the last run_spill."""
        ms = (C.c_double * len(self.STAGES))()
        ln = (C.c_int64 * len(self.STAGES))()
        fma = C.c_double(0.0)
        _check(self.lib.lartpc_get_stage_ms(self.handle, ms, ln, C.byref(fma)), "lartpc_get_stage_ms")
        return dict(zip(self.STAGES, ms)), dict(zip(self.STAGES, ln)), float(fma.value)

    COUNTERS = ("fma_needed", "response_mma", "response_bytes_to_smem", "charge_columns", "charge_mma", "response_items")

    def counters(self):
        """Device-counted S4 work of the last run_spill (lartpc_get_counters)."""
        out = (C.c_double * 8)()
        _check(self.lib.lartpc_get_counters(self.handle, out), "lartpc_get_counters")
        return dict(zip(self.COUNTERS, [float(x) for x in out]))

    def workspace_bytes(self, max_segments: int) -> int:
        return int(self.lib.lartpc_workspace_bytes(self.handle, C.c_int64(max_segments)))

    def run_spill(self, seg, seed: int, hit_capacity: int, workspace=None, hits=None):
        """S7: whole path on device-resident segments.  Returns (hits dict, Stats).  Pass ``workspace``
        (a uint8 CUDA tensor) and ``hits`` (from a previous call) to reuse buffers."""
        t = self.torch
        s, n = self._seg_struct(seg)
        if workspace is None:
            workspace = self._empty(self.workspace_bytes(n), t.uint8)
        if hits is None:
            out, h = self._hits(hit_capacity, None)
            out["_struct"] = h
        else:
            out, h = hits, hits["_struct"]
        st = Stats()
        _check(self.lib.lartpc_run_spill(self.handle, C.byref(s), C.c_int64(n), C.c_uint64(seed), C.byref(h),
                                         C.byref(st), C.c_void_p(workspace.data_ptr()),
                                         C.c_size_t(workspace.numel()), _stream_ptr(t)), "lartpc_run_spill")
        return out, st

    def pack_hits(self, hits, n_hits: Optional[int] = None, tile_pixels: int = 70):
        """16-bit packed hit output grouped by readout tile: returns (packed int16 tensor [n_hits, 3] holding the
        uint16 words, tile_offsets int64 tensor [n_tiles + 1])."""
        t = self.torch
        n = int(hits["counters"][0].item()) if n_hits is None else int(n_hits)
        self.lib.lartpc_readout_tiles.restype = C.c_int64
        n_rt = int(self.lib.lartpc_readout_tiles(self.handle, C.c_int(int(tile_pixels))))
        if n_rt < 0:
            _check(n_rt, "lartpc_readout_tiles")
        packed = self._empty(3 * max(n, 1), t.int16)
        offs = self._empty(n_rt + 1, t.int64)
        _check(self.lib.lartpc_pack_hits(self.handle, C.byref(hits["_struct"]), C.c_int64(n), C.c_int(int(tile_pixels)),
                                         C.c_void_p(packed.data_ptr()), C.c_void_p(offs.data_ptr()), _stream_ptr(t)),
               "lartpc_pack_hits")
        return packed[:3 * n].view(n, 3), offs


class LightSim:
    """Owns a ``lartpc_light_t``: the light look-up table, sensor efficiencies and gains, the impulse
    response and the noise spectrum.  Argument marshalling only; every step runs in the library's kernels."""

    def __init__(self, params: Dict, eff, gain, vis, tprof, resp, noise_amp=None, noise_k=None, device: str = "cuda:0"):
        torch = _torch()
        self.torch = torch
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.lib = load_library()
        self.params = dict(params)
        p = LightParams()
        for name, _ in LightParams._fields_:
            setattr(p, name, params[name])
        f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
        eff, gain, vis, tprof, resp = f32(eff), f32(gain), f32(vis), f32(tprof), f32(resp)
        nd, nvox = int(params["n_det"]), int(params["nvx"]) * int(params["nvy"]) * int(params["nvz"])
        if eff.size != nd or gain.size != nd or vis.size != nd * nvox or tprof.size != nd * nvox * int(params["n_lut_t"]) \
                or resp.size != int(params["n_resp"]):
            raise LartpcError("light tables do not have the sizes the parameters give")
        nn = int(params["n_noise"])
        amp = f32(noise_amp if nn else np.zeros(1))
        nk = np.ascontiguousarray(noise_k if nn else np.zeros(1), dtype=np.int32)
        if nn and (amp.size != nn or nk.size != nn):
            raise LartpcError("noise spectrum does not have n_noise entries")
        ptr = lambda a: a.ctypes.data_as(C.c_void_p)
        h = C.c_void_p()
        _check(self.lib.lartpc_light_create(C.byref(p), ptr(eff), ptr(gain), ptr(vis), ptr(tprof), ptr(resp), ptr(amp), ptr(nk),
                                            C.byref(h)), "lartpc_light_create")
        self.handle = h
        self.n_det, self.n_ticks = nd, int(params["n_ticks"])

    def close(self):
        if getattr(self, "handle", None):
            self.lib.lartpc_light_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _empty(self, n, dtype):
        return self.torch.empty(int(max(n, 1)), dtype=dtype, device=self.device)

    def _wave(self):
        return self.torch.empty((self.n_det, self.n_ticks), dtype=self.torch.float32, device=self.device)

    def _segs(self, seg):
        s = Segments()
        for k in SEG_FIELDS:
            v = seg[k]
            if v.dtype != self.torch.float32 or not v.is_cuda or not v.is_contiguous():
                raise LartpcError("segment field %s must be a contiguous float32 CUDA tensor" % k)
            setattr(s, k, v.data_ptr())
        return s, int(seg["xs"].numel())

    def npe(self, seg, n_e):
        """L1, eqs. (4.1)(4.2): dict(vox, k0, n_gamma [n], npe [n_det, n])."""
        t = self.torch
        s, n = self._segs(seg)
        out = dict(vox=self._empty(n, t.int32), k0=self._empty(n, t.int32), n_gamma=self._empty(n, t.float32),
                   npe=self._empty(self.n_det * n, t.float32))
        _check(self.lib.lartpc_light_npe(self.handle, C.byref(s), C.c_int64(n), C.c_void_p(n_e.data_ptr()),
                                         C.c_void_p(out["vox"].data_ptr()), C.c_void_p(out["k0"].data_ptr()),
                                         C.c_void_p(out["n_gamma"].data_ptr()), C.c_void_p(out["npe"].data_ptr()),
                                         _stream_ptr(t)), "lartpc_light_npe")
        out = {k: v[:n] if k != "npe" else v[:self.n_det * n].view(self.n_det, n) for k, v in out.items()}
        out["_n"] = n
        return out

    def profile(self, a):
        """L2, eq. (4.3): photoelectrons per tick [n_det, n_ticks]."""
        out = self._wave()
        _check(self.lib.lartpc_light_profile(self.handle, C.c_int64(a["_n"]), C.c_void_p(a["vox"].data_ptr()),
                                             C.c_void_p(a["k0"].data_ptr()), C.c_void_p(a["npe"].data_ptr()),
                                             C.c_void_p(out.data_ptr()), _stream_ptr(self.torch)), "lartpc_light_profile")
        return out

    def scintillation(self, ipe):
        out = self._wave()
        _check(self.lib.lartpc_light_scintillation(self.handle, C.c_void_p(ipe.data_ptr()), C.c_void_p(out.data_ptr()),
                                                   _stream_ptr(self.torch)), "lartpc_light_scintillation")
        return out

    def fluctuate(self, isc, seed: int):
        out = self._wave()
        _check(self.lib.lartpc_light_fluctuate(self.handle, C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF), C.c_void_p(isc.data_ptr()),
                                               C.c_void_p(out.data_ptr()), _stream_ptr(self.torch)), "lartpc_light_fluctuate")
        return out

    def electronics(self, nobs, seed: int):
        out = self._wave()
        _check(self.lib.lartpc_light_electronics(self.handle, C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF),
                                                 C.c_void_p(nobs.data_ptr()), C.c_void_p(out.data_ptr()),
                                                 _stream_ptr(self.torch)), "lartpc_light_electronics")
        return out

    def workspace_bytes(self, n: int) -> int:
        return int(self.lib.lartpc_light_workspace_bytes(self.handle, C.c_int64(int(n))))

    def run(self, seg, n_e, seed: int, workspace=None):
        """L1..L5: the read-out waveforms [n_det, n_ticks]."""
        t = self.torch
        s, n = self._segs(seg)
        if workspace is None:
            workspace = t.empty(self.workspace_bytes(n), dtype=t.uint8, device=self.device)
        out = self._wave()
        _check(self.lib.lartpc_light_run(self.handle, C.byref(s), C.c_int64(n), C.c_void_p(n_e.data_ptr()),
                                         C.c_uint64(int(seed) & 0xFFFFFFFFFFFFFFFF), C.c_void_p(out.data_ptr()),
                                         C.c_void_p(workspace.data_ptr()), C.c_size_t(workspace.numel()), _stream_ptr(t)),
               "lartpc_light_run")
        return out


def hits_to_numpy(hits, n: Optional[int] = None):
    """(pixel, tick, adc) int32 numpy arrays of the first ``n`` (default: counters[0]) hits."""
    n = int(hits["counters"][0].item()) if n is None else n
    return (hits["hit_pixel"][:n].cpu().numpy(), hits["hit_tick"][:n].cpu().numpy(), hits["hit_adc"][:n].cpu().numpy())
