"""Helpers of the ``-m gpu`` parity tests: run the CUDA path stage by stage through the C-ABI binding."""
import numpy as np


def run_staged(sim, wl, seed=None):
    """S1..S6 through the staged entry points; returns numpy views of every stage output."""
    import torch
    seg = sim.upload_segments(wl.segments)
    dedx, ne = sim.quench(seg)
    dr = sim.drift(seg, ne)
    pm, info = sim.pixels_from_segments(seg, dr)
    sig = sim.induced_current(dr, pm)
    wf = sim.sum_pixel_signals(sig)
    hits = sim.electronics(wf, wl.seed if seed is None else seed)
    torch.cuda.synchronize()
    cpu = lambda d: {k: v.cpu().numpy() for k, v in d.items() if not k.startswith("_")}
    out = dict(dEdx=dedx.cpu().numpy(), n_e=ne.cpu().numpy(), drift=cpu(dr), pixmap=cpu(pm), info=info,
               waveforms=cpu(wf), hits=cpu(hits))
    out["n_active"] = int(wf["_struct"].n_active)
    return out


def dense_waves(res, n_ticks):
    """[n_active][n_ticks] float64 array from the ragged GPU waveform store."""
    wf = res["waveforms"]
    na = res["n_active"]
    dense = np.zeros((na, n_ticks))
    for i in range(na):
        o, f, l = int(wf["offset"][i]), int(wf["first_tick"][i]), int(wf["length"][i])
        dense[i, f:f + l] = wf["samples"][o:o + l]
    return dense


def hit_table(pix, tick, adc):
    return {(int(p), int(t)): int(a) for p, t, a in zip(pix, tick, adc)}


def compare_hits(gpu, orc):
    """Fraction of oracle hits reproduced exactly, and whether every other hit is off by <= 1 tick or 1 count."""
    g, o = hit_table(*gpu), hit_table(*orc)
    exact = sum(1 for k, a in o.items() if g.get(k) == a)
    near = True
    for (p, t), a in o.items():
        if g.get((p, t)) == a:
            continue
        cands = [g.get((p, t + d)) for d in (-1, 0, 1)]
        if not any(c is not None and abs(c - a) <= 1 for c in cands):
            near = False
    extra = [k for k in g if k not in o and (k[0], k[1] - 1) not in o and (k[0], k[1] + 1) not in o]
    return exact / max(len(o), 1), near and not extra, len(g), len(o)
