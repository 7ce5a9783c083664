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
    """Hit lists compared pixel by pixel, hit by hit, in tick order (BASELINE north_star: >= 99.9 % identical in pixel,
    tick and ADC; the rest off by at most one tick or one count, at threshold crossings).

    A pixel's hits are a chain.  A sample that lands on an ADC code boundary may differ by one count with the tick
    unchanged: the reset is the same, the chain goes on and every later hit is still compared strictly.  When the
    integrated charge sits within the rounding error of the threshold at a crossing, the two sides may fire one tick
    apart; the reset then happens one tick apart, the reset noise is drawn for another (pixel, tick) key and the charge
    of one tick moves between neighbouring samples -- every LATER hit of that pixel is a consequence of that one near
    miss, not an independent disagreement: those are counted as not identical unless they do agree, but not held to the
    nearness rule.  A missing / extra hit without such a near miss before it, or a first difference beyond one tick /
    one count, fails.
    Returns (identical fraction of the oracle's hits, all differences explained, n_gpu, n_oracle, n_near_misses)."""
    def by_pixel(pix, tick, adc):
        d = {}
        for p, t, a in zip(pix.tolist(), tick.tolist(), adc.tolist()):
            d.setdefault(int(p), []).append((int(t), int(a)))
        for v in d.values():
            v.sort()
        return d
    g, o = by_pixel(*gpu), by_pixel(*orc)
    exact = n_o = n_g = n_near = 0
    ok = True
    for p in set(g) | set(o):
        gl, ol = g.get(p, []), o.get(p, [])
        n_o += len(ol)
        n_g += len(gl)
        k = 0
        while k < min(len(gl), len(ol)):
            if gl[k] == ol[k]:
                exact += 1
            elif gl[k][0] == ol[k][0] and abs(gl[k][1] - ol[k][1]) <= 1:
                n_near += 1                     # one count at a code boundary: same tick, same reset, the chain goes on
            else:
                break
            k += 1
        if k == len(gl) == len(ol):
            continue
        if k < min(len(gl), len(ol)) and abs(gl[k][0] - ol[k][0]) <= 1 and abs(gl[k][1] - ol[k][1]) <= 1:
            n_near += 1                         # one tick apart at a crossing; what follows on this pixel is its consequence
            rest = set(gl[k + 1:])
            exact += sum(1 for h in ol[k + 1:] if h in rest)
        else:
            ok = False                          # a missing / extra hit, or a first difference beyond one tick / one count
    return exact / max(n_o, 1), ok, n_g, n_o, n_near
