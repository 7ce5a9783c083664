"""Measurement aid: which (unit of 128 tiles, LUT bin, 16-tick block) operands of the tensor-core response hold charge?

    python -m paper_2212_09807_b200.measure_occupancy [config 2|3]

Runs S1-S4 through the binding with a zero-filled charge buffer, reads the operand image the charge lattice wrote
(include/lartpc.h, lartpc_signals_t.charge) and reports how many (bin, block) operands a tile charges, how many some tile of
each unit charges with the plan's tile order, and what other tile orders would give (simulated on the measured occupancy).
configs[3] is cut down to its two busiest TPCs (the image of the whole spill would not fit beside the workspace).
profiles/r2_response_bound.md holds its output.  Needs a B200 and the built library; no arithmetic of the method here.
"""
from __future__ import annotations

import sys

import numpy as np


def main(cfg: int) -> None:
    import torch
    from . import lartpc, workloads as W

    wl = W.make_config(cfg)
    sim = lartpc.Sim(wl.params, wl.tpcs, wl.lut, response="tensor")
    sim._empty = lambda n, dt: torch.zeros(int(max(n, 0)), dtype=dt, device=sim.device)   # unwritten operands read as zero
    if cfg == 3:
        seg = sim.upload_segments(wl.segments)
        _, ne = sim.quench(seg)
        tpc_of = sim.drift(seg, ne)["tpc"].cpu().numpy()
        counts = np.bincount(tpc_of[tpc_of >= 0], minlength=len(wl.tpcs))
        busy = [int(x) for x in np.argsort(counts)[-2:]]
        wl = wl.subset(np.nonzero(np.isin(tpc_of, busy))[0])
        del seg, ne
    seg = sim.upload_segments(wl.segments)
    _, ne = sim.quench(seg)
    dr = sim.drift(seg, ne)
    pm, info = sim.pixels_from_segments(seg, dr)
    sig = sim.induced_current(dr, pm)
    torch.cuda.synchronize()
    nt, nb2 = int(info.n_tiles), int(wl.params["bins_per_pixel"]) ** 2
    nu = (nt + 127) // 128
    ch = sig["charge"].view(torch.uint8)
    # fp16 part of the image: [unit, bin, block, part 0, 8-row group, row in group, 32 bytes]
    img = ch[: nu * nb2 * 4 * 8192].view(nu, nb2, 4, 2, 16, 8, 32)[:, :, :, 0]
    nzr = (img != 0).any(dim=-1).reshape(nu, nb2, 4, 128)                     # [unit, bin, block, tile row]
    unit_blk = nzr.any(dim=3).any(dim=1)
    union = nzr.any(dim=3)
    tile_blk = nzr.any(dim=1)
    dense_now, dense_cb = int(unit_blk.sum()) * nb2, int(union.sum())
    print("config %d: %d tiles, %d units" % (cfg, nt, nu))
    print("(unit, bin, block) operands in the units' block masks: %d; charged by some tile (the plan's order): %d = %.3f"
          % (dense_now, dense_cb, dense_cb / dense_now))
    print("per tile: (bin, block) pairs charged / bins x blocks charged = %.3f; bins charged %.1f of %d"
          % (int(nzr.sum()) / (int(tile_blk.sum()) * nb2), nzr.any(dim=2).sum(dim=1).float().mean().item(), nb2))
    if nb2 != 100:
        return
    # other tile orders, simulated: sort the tiles by a key, cut into units of 128, count the operands some tile charges
    T = nzr.permute(0, 3, 1, 2).reshape(nu * 128, 100, 4)[:nt]
    bm = (T.any(dim=1).long() * torch.tensor([1, 2, 4, 8], device=T.device)).sum(dim=1)
    occ = T.any(dim=2).reshape(nt, 10, 10)
    idx = torch.arange(10, device=T.device)

    def lo_hi(o):
        return (torch.where(o, idx, 99).min(dim=1).values.clamp(0, 9), torch.where(o, idx, -1).max(dim=1).values.clamp(0, 9))

    alo, ahi = lo_hi(occ.any(dim=1))
    blo, bhi = lo_hi(occ.any(dim=2))
    print("box of charged bins: mean area %.1f" % ((ahi - alo + 1) * (bhi - blo + 1)).float().mean().item())

    def simulate(key, name):
        ts = T[torch.argsort(key, stable=True)]
        pad = (-nt) % 128
        if pad:
            ts = torch.cat([ts, torch.zeros(pad, 100, 4, dtype=torch.bool, device=T.device)])
        u = ts.reshape(-1, 128, 100, 4).any(dim=1)
        print("%-52s %9d operands = %.3f of the plan's block masks" % (name, int(u.sum()), int(u.sum()) / dense_now))

    simulate(bm, "sorted by block mask")
    simulate(bm * 10000 + alo * 1000 + ahi * 100 + blo * 10 + bhi, "by block mask and exact box")
    for q in (2, 3):
        simulate(bm * 10000 + (alo // q) * 1000 + (ahi // q) * 100 + (blo // q) * 10 + bhi // q,
                 "by block mask and box edges in steps of %d bins" % q)
    # more of the pattern in the key: which way the charged bins lean (a track's direction across the pixel), how full the box is
    of = occ.float()
    cnt = of.sum(dim=(1, 2)).clamp(min=1.0)
    ia, ib = idx.float().view(1, 10, 1), idx.float().view(1, 1, 10)
    # occ is [tile][b][a] or [tile][a][b]: the sign of the covariance is the same either way
    ma, mb = (of * ia).sum(dim=(1, 2)) / cnt, (of * ib).sum(dim=(1, 2)) / cnt
    cov = (of * ia * ib).sum(dim=(1, 2)) / cnt - ma * mb
    lean = torch.where(cov > 0.5, 1, torch.where(cov < -0.5, 2, 0))
    area = ((ahi - alo + 1) * (bhi - blo + 1)).float()
    fill = (3.0 * (cnt / area).clamp(max=0.999)).long()
    box2 = (alo // 2) * 1000 + (ahi // 2) * 100 + (blo // 2) * 10 + bhi // 2
    simulate((bm * 10000 + box2) * 3 + lean, "by block mask, box in steps of 2 and lean of the pattern")
    simulate(((bm * 10000 + box2) * 3 + lean) * 3 + fill, "... and how full the box is (3 levels)")
    # the pattern itself as the key (columns of bins, most significant first): identical patterns meet, similar ones mostly do
    colbits = (occ.long() * (1 << idx.long()).view(1, 1, 10)).sum(dim=2)                      # [tile][10] ten-bit words
    key = bm.clone()
    for c in range(10):
        key = key * 1024 + colbits[:, c]
        if c == 4:                                                    # (two 50-bit halves: sort by the second, then stably by the first)
            key_hi, key = key, torch.zeros_like(bm)
    order = torch.argsort(key, stable=True)
    order = order[torch.argsort(key_hi[order], stable=True)]
    ts = T[order]
    pad = (-nt) % 128
    if pad:
        ts = torch.cat([ts, torch.zeros(pad, 100, 4, dtype=torch.bool, device=T.device)])
    u = ts.reshape(-1, 128, 100, 4).any(dim=1)
    print("%-52s %9d operands = %.3f of the plan's block masks" % ("by block mask and the pattern read as a number", int(u.sum()), int(u.sum()) / dense_now))
    sim.close()


if __name__ == "__main__":
    main(int(sys.argv[1]) if len(sys.argv) > 1 else 3)
