// S4  induced current, eqs. (3.7)-(3.9) P:L660-687 with the M-sum in expectation (D1).
//
// Decomposition: the paper's kernel gives one thread to every (segment, pixel, tick)
// and lets it sum N*M LUT look-ups.  By linearity of eq. (3.7) the same sum is
//     C[b][a][j]  = sum_seg sum_mu (Q_a/N) wx[a] wy[b] wt[j]          (charge per LUT cell, eq. 3.8)
//     I_p[n]      = sum_{a,b,j} C[b][a][j] * R[b - nb(iy-H)][a - nb(ix-H)][n - j]      (eq. 3.7)
// which needs ~50x fewer operations and shares the charge lattice between neighbouring segments.
// A tile is (charged pixel P, window of Jc arrival ticks).  Two kernels per path:
//
// Tensor-core path (default; charge_tc.cuh + response_tc.cuh): both factors are dense contractions on tcgen05.
//   charge_lattice_tc_kernel  C = WXY WT^T over the operand columns (node-rule nodes or sample midpoints, or the perturbed
//                             points of eq. (3.9) as printed) of a tile's segments; persistent CTAs, TMEM accumulator,
//                             cp.async look-ahead for descriptors / ids / per-segment records.
//   response_tc_kernel        I = C x Toeplitz(R): per (128-tile block, target, bin) the charged 16-tick blocks of the
//                             operand image against one 16 x NBW LUT generator, fp16 main term + fp8 cross terms.
//
// FFMA2 path (this file; on request or when the window is wider than 11 pixels; FFMA2 charge lattice also for bins per pixel other than 5 / 10):
//   charge_lattice_kernel (one CTA per tile)
//     splat the tile's segments into C[nb*nb][Jc] in shared memory (register-tiled outer products of
//     per-sample erf-difference weights, no atomics, fixed order), then pack the non-empty bins: per bin the
//     first charged tick rounded down to even, the number of 4-tick charge groups and the charge row.
//
//   response_kernel (persistent, two CTAs per SM, no CTA-wide barrier after start-up)
//     warp 8 is the producer: it takes tiles from a work counter and, per non-empty bin, streams the bin's
//     LUT rows (one contiguous block, pair-interleaved targets) and its charge row into a ring of shared-memory
//     stages with cp.async.bulk (TMA engine), completion on an mbarrier per stage.
//     Warps 0-7 are consumers (two per SM sub-partition): a thread owns RESP_NO = 14 output ticks of a PAIR of
//     target pixels (28 accumulators as 14 packed f32x2 registers) for the whole tile and slides a 20-tap window of
//     the pair-interleaved LUT row over the charge row, 4 charges per step: 56 FFMA2 (112 multiply-adds) per
//     2 LDS.128 of taps + 1 broadcast LDS.128 of charge.  Warps run freely through the ring (full / empty
//     mbarriers), so threads with edge output blocks never hold back the others, and the output blocks are dealt
//     to the thread slots so that the four sub-partitions carry the same load (api.cu balance_blocks).  After the
//     last bin of a tile the accumulators go to global memory as the tile's partial waveforms; S5 sums them per
//     pixel in a fixed order.
#include <string.h>
#include <algorithm>
#include "common.cuh"
#include "response_tc.cuh"

namespace {

typedef unsigned long long u64;   // one packed f32x2 register pair: (target 2p, target 2p+1)

__device__ __forceinline__ u64 pack2(float x)
{
    u64 r;
    asm("mov.b64 %0, {%1, %1};" : "=l"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ void ffma2(u64 &d, u64 a, u64 b)      // d = a * b + d on both halves
{
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}

// ---- mbarrier + bulk copy (TMA engine) -------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(void *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(void *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(void *bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    return ok != 0;
}
// the whole warp waits, one lane polls (32 lanes polling one mbarrier serialise in the shared-memory pipe)
__device__ __forceinline__ void mbar_wait_warp(void *bar, uint32_t parity, int lane)
{
    while (true) {
        bool ok = false;
        if (lane == 0) ok = mbar_try_wait(bar, parity);
        if (__any_sync(0xffffffffu, ok)) break;
    }
}
__device__ __forceinline__ bool mbar_try_wait_u32(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_arrive(void *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(void *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// global -> shared bulk copy, completion counted in bytes on `bar`
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, void *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// =====================================================================================================
// Kernel 1: charge lattice of every tile
// =====================================================================================================
constexpr int NT1 = 256;         // threads per CTA
constexpr int SB = 64;           // samples per splat batch
constexpr int XS = 16;           // row length of the per-sample x / y weight tables (bins_per_pixel <= 15)
constexpr int SEGCAP = 32;       // segments staged per batch

struct SplatArgs {
    DevParams p;
    const DevTpc *tpcs;
    const int32_t *tile_cp;
    const TileDesc *tile_desc;
    const int32_t *pix_start, *pix_count, *pair_seg;
    const float *q_anode, *sigma_T, *sigma_t;
    const double *u_s, *v_s, *u_e, *v_e, *T_s, *T_e;
    const int32_t *a_lo, *a_hi, *b_lo, *b_hi, *jt0, *jt1, *n_samples;
    float *charge;                     // [n_tiles][slab_floats]
    int32_t *tile_range;
    unsigned long long *fma_counter;   // multiply-adds of the response: non-zero cells x valid targets x K
    // tensor-core splat (charge_tc.cuh): persistent CTAs
    const void *rec;                   // SegRec[n]
    const int2 *tile_list;             // [n_tiles] {start, count} of the tile's segment list in pair_seg
    int *work;                         // tile cursor, zero at launch
    int n_tiles;
    const int32_t *tb_mask;            // [tile blocks] 16-tick blocks that hold charge (bit b)
    int32_t *cmask;                    // [units][TC_CMASK_WORDS] per LUT bin the blocks some tile of the unit charges (tensor-core splat)
};

struct SegLocal {               // one staged segment, tile-relative
    float as, ae, bs, be, ts, te, isT, ist, q;
    int N, alo, ahi, blo, bhi, jlo, jhi, seg, zero_sigma;
    float qa, inv_n2, inv_n4;   // tensor-core splat: Q_a and 1/N^2, 1/N^4 of the node-rule weights (charge_tc.cuh)
    int rule;                   // first row of the segment's node rule in g_quad, -1: its own N midpoints
};

__global__ void __launch_bounds__(NT1, 3) charge_lattice_kernel(const SplatArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NB2 = p.NB2, CJ = p.CJ, nb = p.nb, K = p.K;

    float *Csm = (float *)smem_raw;                                  // [NB2][CJ] charge per (bin, arrival tick)
    float *scratch = Csm + NB2 * CJ;                                 // splat scratch
    int *s_int = (int *)(scratch + SB * (2 * XS + CJ));
    int *bin_jlo = s_int, *bin_jhi = s_int + NB2, *bin_list = s_int + 2 * NB2, *bin_off = s_int + 3 * NB2;
    int *s_misc = s_int + 4 * NB2;                                   // [0] n bins, [1] tile jlo, [2] tile jhi, [3] groups
    SegLocal *segs = (SegLocal *)(s_misc + 8);

    const int tile = blockIdx.x;
    const TileDesc td = a.tile_desc[tile];
    const int cp = a.tile_cp[tile];
    const DevTpc &tp = a.tpcs[td.tpc];
    const int A_t = td.px * nb, B_t = td.py * nb, J_t = td.j_start;
    const int lstart = a.pix_start[cp], lcount = a.pix_count[cp];

    for (int i = tid; i < NB2 * CJ / 4; i += NT1) ((float4 *)Csm)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

    // ------------------------------------------------------------------ phase 1: splat
    float *WX = scratch, *WY = scratch + SB * XS, *WT = scratch + 2 * SB * XS;     // [SB][XS], [SB][XS], [SB][CJ]
    for (int l0 = 0; l0 < lcount; l0 += SEGCAP) {
        __syncthreads();
        const int nseg = min(SEGCAP, lcount - l0);
        if (tid < nseg) {
            const int s = a.pair_seg[lstart + l0 + tid];
            SegLocal L;
            L.seg = s;
            L.N = a.n_samples[s];
            L.alo = max(a.a_lo[s] - A_t, 0);  L.ahi = min(a.a_hi[s] - A_t, nb - 1);
            L.blo = max(a.b_lo[s] - B_t, 0);  L.bhi = min(a.b_hi[s] - B_t, nb - 1);
            L.jlo = max(max(a.jt0[s], 0) - J_t, 0);
            L.jhi = min(min(a.jt1[s], p.j_max) - J_t, p.Jc - 1);
            const double inv_bin = 1.0 / p.bin, inv_dt = 1.0 / p.dt;
            L.as = (float)(a.u_s[s] * inv_bin - (double)A_t);  L.ae = (float)(a.u_e[s] * inv_bin - (double)A_t);
            L.bs = (float)(a.v_s[s] * inv_bin - (double)B_t);  L.be = (float)(a.v_e[s] * inv_bin - (double)B_t);
            L.ts = (float)((a.T_s[s] - p.t_origin) * inv_dt - (double)J_t);
            L.te = (float)((a.T_e[s] - p.t_origin) * inv_dt - (double)J_t);
            const float sT = a.sigma_T[s], st = a.sigma_t[s];
            L.zero_sigma = !(sT > 0.0f) || !(st > 0.0f);
            L.isT = L.zero_sigma ? 0.f : (float)(p.bin * 0.70710678118654752440 / (double)sT);
            L.ist = L.zero_sigma ? 0.f : (float)(p.dt * 0.70710678118654752440 / (double)st);
            L.q = a.q_anode[s] / (float)L.N;                          // eq. (3.8): Q_a / N per sample point
            segs[tid] = L;
        }
        __syncthreads();
        for (int li = 0; li < nseg; ++li) {
            const SegLocal L = segs[li];
            if (L.jlo > L.jhi || L.alo > L.ahi || L.blo > L.bhi) continue;          // CTA-uniform
            if (L.zero_sigma) {
                // sigma = 0: the weights are indicators; the bin / tick is an integer decision taken in
                // float64 with the oracle's operation order (SURVEY section 7 "sigma -> 0 branch")
                const int s = L.seg;
                const double us = a.u_s[s], ue = a.u_e[s], vs = a.v_s[s], ve = a.v_e[s], Ts = a.T_s[s], Te = a.T_e[s];
                for (int mu = tid; mu < L.N; mu += NT1) {
                    double f = xdiv(xadd((double)mu, 0.5), (double)L.N);
                    double u = xadd(us, xmul(xsub(ue, us), f));
                    double v = xadd(vs, xmul(xsub(ve, vs), f));
                    double T = xadd(Ts, xmul(xsub(Te, Ts), f));
                    long long ia = (long long)floor(xdiv(u, p.bin)) - A_t, ib = (long long)floor(xdiv(v, p.bin)) - B_t;
                    long long j = (long long)floor(xdiv(xsub(T, p.t_origin), p.dt));
                    if (j < 0 || j > p.j_max) continue;
                    j -= J_t;
                    if (ia >= 0 && ia < nb && ib >= 0 && ib < nb && j >= 0 && j < p.Jc)
                        atomicAdd(&Csm[((int)ib * nb + (int)ia) * CJ + (int)j], L.q);
                }
                __syncthreads();
                continue;
            }
            const int na = L.ahi - L.alo + 1, nbb = L.bhi - L.blo + 1, nj = L.jhi - L.jlo + 1;
            const int na4 = (na + 3) >> 2, nj4 = (nj + 3) >> 2, units = na4 * nbb * nj4;
            const int truns = (nj + 30) / 31, runs = 1 + truns;       // warp runs per sample: (x | y) and the t pieces
            const float invN = 1.0f / (float)L.N;
            const int npass = (L.N + SB - 1) / SB, nsb_max = (L.N + npass - 1) / npass;
            for (int mu0 = 0; mu0 < L.N; mu0 += nsb_max) {
                const int nsb = min(nsb_max, L.N - mu0);
                // (A) one-dimensional cell weights of every sample of the batch.  A warp evaluates erf once per bin /
                // tick edge and takes the difference with its neighbour lane: w = (erf(e+1) - erf(e)) / 2.
                for (int r = warp; r < nsb * runs; r += NT1 / 32) {
                    const int ml = r / runs, k = r - ml * runs;
                    const float f = ((float)(mu0 + ml) + 0.5f) * invN;
                    if (k == 0) {
                        const int half = lane >> 4, e = lane & 15;     // lanes 0-15: x edges, 16-31: y edges
                        const float pos = half ? fmaf(L.be - L.bs, f, L.bs) : fmaf(L.ae - L.as, f, L.as);
                        const float E = erff(((float)((half ? L.blo : L.alo) + e) - pos) * L.isT);
                        const float En = __shfl_down_sync(0xffffffffu, E, 1);
                        if (e < (half ? nbb : na)) (half ? WY : WX)[ml * XS + e] = 0.5f * (En - E);
                    } else {
                        const int e = 31 * (k - 1) + lane;            // 32 edges -> 31 weights per run
                        const float pos = fmaf(L.te - L.ts, f, L.ts);
                        const float E = erff(((float)(L.jlo + e) - pos) * L.ist);
                        const float En = __shfl_down_sync(0xffffffffu, E, 1);
                        if (lane < 31 && e < nj) WT[ml * CJ + e] = 0.5f * L.q * (En - E);
                    }
                }
                __syncthreads();
                // (B) a thread owns 4 cells (consecutive in a) x 4 ticks and adds the batch's outer products to them;
                // entries past na / nj multiply stale shared memory and are never stored
                for (int unit = tid; unit < units; unit += NT1) {
                    const int cu = unit / nj4, jq = unit - cu * nj4, b = cu / na4, aq = cu - b * na4;
                    u64 acc[4][2];
#pragma unroll
                    for (int i = 0; i < 4; ++i) acc[i][0] = acc[i][1] = 0ull;
                    const float *px = WX + aq * 4, *py = WY + b, *pt = WT + jq * 4;
#pragma unroll 2
                    for (int ml = 0; ml < nsb; ++ml) {
                        const float4 x4 = *(const float4 *)(px + ml * XS);
                        const float y = py[ml * XS];
                        const ulonglong2 t4 = *(const ulonglong2 *)(pt + ml * CJ);
                        const float w[4] = {x4.x * y, x4.y * y, x4.z * y, x4.w * y};
#pragma unroll
                        for (int i = 0; i < 4; ++i) {
                            ffma2(acc[i][0], pack2(w[i]), t4.x);
                            ffma2(acc[i][1], pack2(w[i]), t4.y);
                        }
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        if (aq * 4 + i < na) {
                            float *row = Csm + ((L.blo + b) * nb + (L.alo + aq * 4 + i)) * CJ + L.jlo + jq * 4;
                            const float v[4] = {__uint_as_float((unsigned)acc[i][0]), __uint_as_float((unsigned)(acc[i][0] >> 32)),
                                                __uint_as_float((unsigned)acc[i][1]), __uint_as_float((unsigned)(acc[i][1] >> 32))};
#pragma unroll
                            for (int k = 0; k < 4; ++k)
                                if (jq * 4 + k < nj) row[k] += v[k];
                        }
                    }
                }
                __syncthreads();
            }
        }
    }
    __syncthreads();

    // ------------------------------------------------------------------ phase 2: non-empty bins and their tick ranges
    int nz_cells = 0;
    for (int c = warp; c < NB2; c += NT1 / 32) {
        int lo = INT_MAX, hi = -1;
        for (int j = lane; j < p.Jc; j += 32)
            if (Csm[c * CJ + j] != 0.f) { lo = min(lo, j); hi = max(hi, j); ++nz_cells; }
        for (int d = 16; d; d >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, d));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, d));
        }
        if (lane == 0) { bin_jlo[c] = lo; bin_jhi[c] = hi; }
    }
    __syncthreads();
    if (warp == 0) {
        // bin list in ascending bin order; row offsets = running sum of 4 * groups
        // (rows are copied by 16-byte bulk transfers: the first one starts on a multiple of four words)
        int nbins = 0, tlo = INT_MAX, thi = -1, off = (SLAB_HDR + 2 * NB2 + 3) & ~3, groups = 0;
        for (int base = 0; base < NB2; base += 32) {
            const int c = base + lane;
            const bool f = c < NB2 && bin_jhi[c] >= 0;
            const unsigned bal = __ballot_sync(0xffffffffu, f);
            const int ng = f ? ((bin_jhi[c] - (bin_jlo[c] & ~1)) >> 2) + 1 : 0;
            int inc = f ? ng + 1 : 0;                                // inclusive warp scan of the row lengths in 16-byte units
            for (int d = 1; d < 32; d <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, inc, d);
                if (lane >= d) inc += o;
            }
            if (f) {
                const int k = nbins + __popc(bal & ((1u << lane) - 1u));
                bin_list[k] = c;
                bin_off[k] = off + 4 * (inc - ng - 1);
                tlo = min(tlo, bin_jlo[c]);  thi = max(thi, bin_jhi[c]);
            }
            const int tot = __shfl_sync(0xffffffffu, inc, 31);
            off += 4 * tot;  groups += tot - __popc(bal);
            nbins += __popc(bal);
        }
        for (int d = 16; d; d >>= 1) {
            tlo = min(tlo, __shfl_xor_sync(0xffffffffu, tlo, d));
            thi = max(thi, __shfl_xor_sync(0xffffffffu, thi, d));
        }
        if (lane == 0) { s_misc[0] = nbins; s_misc[1] = tlo; s_misc[2] = thi; s_misc[3] = groups; }
    }
    __syncthreads();
    const int nbins = s_misc[0], tjlo = s_misc[1], tjhi = s_misc[2];
    float *slab = a.charge + (size_t)tile * p.slab_floats;
    int *slab_i = (int *)slab;
    if (nbins == 0) {
        // no charge: S5 skips the tile (first block > last block); the tensor-core response still multiplies whatever
        // the tile's operand rows hold, and nobody reads the result
        if (tid == 0) {
            if (!p.tc_mode) { slab_i[0] = 0; slab_i[1] = 0; slab_i[2] = 1; slab_i[3] = 0; }
            *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(1, 0, 0, 0);
        }
        if (!p.tc_mode) return;
    }
    if (nbins) {
        // multiply-adds the method needs here: non-zero cells x in-plane targets x K
        for (int d = 16; d; d >>= 1) nz_cells += __shfl_xor_sync(0xffffffffu, nz_cells, d);
        const int vx = min(td.px + p.H, tp.nx - 1) - max(td.px - p.H, 0) + 1;
        const int vy = min(td.py + p.H, tp.ny - 1) - max(td.py - p.H, 0) + 1;
        if (lane == 0 && nz_cells && vx > 0 && vy > 0)
            atomicAdd(a.fma_counter, (unsigned long long)nz_cells * (unsigned long long)(vx * vy * K));
    }

    // ------------------------------------------------------------------ phase 3: tile out
    const int nB_lo = tjlo / RESP_NO, nB_hi = (tjhi + K - 1) / RESP_NO; // output blocks, tile-relative
    if (p.tc_mode) {
        // Tensor-core operand image (response_tc.cuh): C * 2^-e split into fp16 hi + lo, row (tile % 128) of the
        // 128-byte-swizzled K-major [128 x 64] block of every bin; e keeps the largest cell below 2^15.
        float mx = 0.f;
        for (int i = tid; i < NB2 * CJ; i += NT1) mx = fmaxf(mx, fabsf(Csm[i]));
        for (int d = 16; d; d >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        __syncthreads();                                                  // scratch is free: the splat is over
        if (lane == 0) scratch[warp] = mx;
        __syncthreads();
        mx = scratch[0];
#pragma unroll
        for (int w = 1; w < NT1 / 32; ++w) mx = fmaxf(mx, scratch[w]);
        int e = 0;
        if (mx >= 32768.f) e = min(((__float_as_int(mx) >> 23) & 0xff) - 127 - 14, 100);   // mx * 2^-e in [2^14, 2^15)
        if (!(mx < 3.0e38f)) e = 0;                                       // inf / nan charge: leave it visible
        const float sc = __int_as_float((127 - e) << 23);
        if (tid == 0 && nbins) *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(nB_lo, nB_hi, e, 0);
        const int tb = tile / rtc::TB, r = tile - tb * rtc::TB;
        unsigned char *Ab = (unsigned char *)a.charge + (size_t)tb * NB2 * (rtc::NBLK * rtc::A_BLOCK_BYTES);
        for (int item = tid; item < NB2 * rtc::NBLK; item += NT1) {
            const int c = item / rtc::NBLK, b = item - c * rtc::NBLK;
            float x[16];
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = Csm[c * CJ + 16 * b + i] * sc;
            rtc::store_a_block16(Ab + ((size_t)c * rtc::NBLK + b) * rtc::A_BLOCK_BYTES, r, x);
        }
        return;
    }
    if (tid == 0) {
        slab_i[0] = nbins; slab_i[1] = s_misc[3]; slab_i[2] = nB_lo; slab_i[3] = nB_hi;
        *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(nB_lo, nB_hi, 0, 0);
    }
    for (int k = tid; k < nbins; k += NT1) {
        const int c = bin_list[k], jb0 = bin_jlo[c] & ~1, ng = ((bin_jhi[c] - jb0) >> 2) + 1;
        slab_i[SLAB_HDR + 2 * k] = c | (ng << 8) | (jb0 << 16);
        slab_i[SLAB_HDR + 2 * k + 1] = bin_off[k];
    }
    // a row = 16-byte header {first charged tick, groups, flags, tile} + 4 * groups charges; the response kernel copies
    // it into a pipeline stage as it is
    const int row_flags = (nB_lo << 8) | (nB_hi << 16);
    for (int k = warp; k < nbins; k += NT1 / 32) {
        const int c = bin_list[k], jb0 = bin_jlo[c] & ~1, ng = ((bin_jhi[c] - jb0) >> 2) + 1;
        const float4 *src = (const float4 *)(Csm + c * CJ + jb0);     // CJ and jb0 even, rows padded by 4 zeros:
        float4 *dst = (float4 *)(slab + bin_off[k]);                  // 8-byte aligned source, 16-byte aligned target
        if (lane == 0) *(int4 *)dst = make_int4(jb0, ng, row_flags | (k == nbins - 1 ? 1 : 0), tile);
        for (int g = lane; g < ng; g += 32) {
            const float2 x = ((const float2 *)src)[2 * g], y = ((const float2 *)src)[2 * g + 1];
            dst[1 + g] = make_float4(x.x, x.y, y.x, y.y);
        }
    }
}

#include "quadrature_tables.cuh"
#include "charge_tc.cuh"
#include "truth.cuh"

size_t splat_smem_bytes(const DevParams &p)
{
    size_t floats = (size_t)p.NB2 * p.CJ + (size_t)SB * (2 * XS + p.CJ);
    size_t ints = 4 * (size_t)p.NB2 + 8;
    size_t bytes = (floats + ints) * 4;
    bytes = (bytes + 15) & ~(size_t)15;
    return bytes + sizeof(SegLocal) * SEGCAP;
}

// =====================================================================================================
// Kernel 2: response of the W x W pixels around every tile (persistent, warp-specialised)
// =====================================================================================================
constexpr int NCW = RESP_CONSUMERS / 32;   // consumer warps
constexpr int NT2 = RESP_CONSUMERS + 32;   // threads per CTA: 8 consumer warps + 1 producer warp, two CTAs per SM
constexpr int NO = RESP_NO;                // output ticks per response task
constexpr int FLAG_LAST = 1, FLAG_END = 2;

struct ResponseArgs {
    DevParams p;
    const float *lut;            // [NB2][NP][RS][2]
    const float *charge;         // [n_tiles][slab_floats]
    float *partial;              // [n_tiles][WW][tile_ticks]
    int *work;                   // work-queue cursor
    int n_work;                  // n_tiles * n_groups
    int n_stages;
    int stage_floats;            // LUT block + charge row + header, in floats (multiple of 4)
    int lut_floats;              // PG * RS * 2
    const int *end_row;          // 16 bytes: a row header with FLAG_END
    unsigned char blk_of_slot[256];
};

__device__ __forceinline__ void load4w(u64 (&d)[4], const float *s)     // 4 pair-words = 32 bytes
{
    const ulonglong2 v0 = *(const ulonglong2 *)s, v1 = *(const ulonglong2 *)(s + 4);
    d[0] = v0.x; d[1] = v0.y; d[2] = v1.x; d[3] = v1.y;
}
__device__ __forceinline__ void load4c(u64 (&c)[4], const float *s)     // 4 charges, each duplicated into a pair
{
    const float4 x = *(const float4 *)s;
    c[0] = pack2(x.x); c[1] = pack2(x.y); c[2] = pack2(x.z); c[3] = pack2(x.w);
}
// acc[i] += sum_jj c[jj] * w[i - jj + 4],  w = q0[0..3] ++ q1 ++ q2 ++ q3 ++ q4  (i < 16, jj < 4)
__device__ __forceinline__ void fma_step(u64 (&acc)[NO], const u64 (&c)[4], const u64 (&q0)[4], const u64 (&q1)[4],
                                         const u64 (&q2)[4], const u64 (&q3)[4], const u64 (&q4)[4])
{
#pragma unroll
    for (int jj = 0; jj < 4; ++jj)
#pragma unroll
        for (int i = 0; i < NO; ++i) {
            const int m = i - jj + 4;
            ffma2(acc[i], c[jj], m < 4 ? q0[m] : (m < 8 ? q1[m - 4] : (m < 12 ? q2[m - 8] : (m < 16 ? q3[m - 12] : q4[m - 16]))));
        }
}

#ifdef LARTPC_DEBUG_CLOCKS
__device__ unsigned long long g_dbg[8];
#define DBG_T(x) long long x = clock64()
#define DBG_ADD(i, v) dbg_acc[i] += (unsigned long long)(v)
#define DBG_DECL unsigned long long dbg_acc[4] = {0, 0, 0, 0}
#define DBG_FLUSH do { if (lane == 0) for (int i_ = 0; i_ < 4; ++i_) atomicAdd(&g_dbg[i_], dbg_acc[i_]); } while (0)
#else
#define DBG_T(x)
#define DBG_ADD(i, v)
#define DBG_DECL
#define DBG_FLUSH
#endif

__global__ void __launch_bounds__(NT2, 2) response_kernel(const ResponseArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int S = a.n_stages;
    float *stages = (float *)smem_raw;                                // [S][stage_floats]: LUT rows, charge row, header
    u64 *full = (u64 *)(stages + (size_t)S * a.stage_floats);        // [S] "stage filled" (1 arrival + bytes)
    u64 *empty = full + S;                                            // [S] "stage released" (NCW arrivals); then int[S]: pair group

    if (tid == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NCW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NCW) {
        // ------------------------------------------------------------------ producer: one thread, few instructions per
        // bin (it shares its sub-partition's issue port with four consumer warps)
        if (lane != 0) return;
        int s = 0;
        uint32_t ph = 0;
        const uint32_t lut_bytes = (uint32_t)a.lut_floats * 4u, stage_bytes = (uint32_t)a.stage_floats * 4u;
        const uint32_t stage0 = smem_u32(stages), full0 = smem_u32(full), empty0 = smem_u32(empty);
        const size_t lut_bin_stride = (size_t)p.NP * p.RS * 2;
        int q = atomicAdd(a.work, 1), q_next = atomicAdd(a.work, 1);
        while (q < a.n_work) {
            const int tile = q / p.n_groups, g = q - tile * p.n_groups;
            const float *slab = a.charge + (size_t)tile * p.slab_floats;
            const int nbins = *(const int *)slab;
            const int2 *items = (const int2 *)(slab + SLAB_HDR);
            const float *lut_g = a.lut + (size_t)g * a.lut_floats;
            int4 nxt = *(const int4 *)items;                         // two items per 16-byte load, one pair ahead
            for (int k = 0; k < nbins; k += 2) {
                const int4 cur = nxt;
                if (k + 2 < nbins) nxt = *(const int4 *)(items + k + 2);
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    if (k + e >= nbins) break;
                    const int w0 = e ? cur.z : cur.x, off = e ? cur.w : cur.y;
                    const int c = w0 & 0xff, ng = (w0 >> 8) & 0xff;
                    const uint32_t st = stage0 + (uint32_t)s * stage_bytes, fb = full0 + 8u * s;
                    const uint32_t row_bytes = 16u + (uint32_t)ng * 16u;
                    while (!mbar_try_wait_u32(empty0 + 8u * s, ph ^ 1u)) {}
                    ((volatile int *)(empty + S))[s] = g;                      // pair group of the stage (released by the arrive below)
                    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"(lut_bytes + row_bytes) : "memory");
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(st), "l"(lut_g + (size_t)c * lut_bin_stride), "r"(lut_bytes), "r"(fb) : "memory");
                    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                 ::"r"(st + lut_bytes), "l"(slab + off), "r"(row_bytes), "r"(fb) : "memory");
                    if (++s == S) { s = 0; ph ^= 1u; }
                }
            }
            q = q_next;
            q_next = atomicAdd(a.work, 1);
        }
        {                                                            // terminator: a header-only row with the END flag
            const uint32_t st = stage0 + (uint32_t)s * stage_bytes, fb = full0 + 8u * s;
            while (!mbar_try_wait_u32(empty0 + 8u * s, ph ^ 1u)) {}
            asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(fb), "r"(16u) : "memory");
            asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                         ::"r"(st + lut_bytes), "l"(a.end_row), "r"(16u), "r"(fb) : "memory");
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    const int slot = tid / p.PG, pl = tid - slot * p.PG;
    const bool valid = slot < p.nblk_max;
    const int blk = valid ? a.blk_of_slot[slot] : 0;
    const int n0 = NO * blk;
    const int K = p.K, WW = p.WW;
    // float offset of pair-word (LUT_OFF + n0 - 4) of this thread's pair row inside a stage; m-range constants
    const int tap0 = (pl * p.RS + (LUT_OFF + n0 - 4)) * 2;
    const int lo_num = n0 - K - 2 + 3, hi_num = n0 + NO - 1;
    const uint32_t full0 = smem_u32(full), empty0 = smem_u32(empty);
    u64 acc[NO];
#pragma unroll
    for (int i = 0; i < NO; ++i) acc[i] = 0ull;
    int s = 0;
    uint32_t ph = 0;
    DBG_DECL;
    while (true) {
        const float *st = stages + (size_t)s * a.stage_floats;
        DBG_T(t0);
        while (!mbar_try_wait_u32(full0 + 8u * s, ph)) {}
        DBG_T(t1);
        DBG_ADD(0, t1 - t0);
        DBG_ADD(3, 1);
        const float *row = st + a.lut_floats;
        const int4 h = *(const int4 *)row;                            // first charged tick, groups, flags, tile
        const int g = ((volatile int *)(empty + S))[s];              // pair group of this pass, published by the producer
        if ((h.z & FLAG_END) | (g < 0)) { DBG_FLUSH; break; }
        if (valid) {
            const int jb0 = h.x, ng = h.y;
            // group m holds charges j = jb0 + 4m .. + 3; its taps k = n - j meet [0, K) for this task's outputs when
            int m = max(0, (lo_num - jb0) >> 2);
            const int m_hi = min(ng - 1, (hi_num - jb0) >> 2);
            if (m <= m_hi) {
                // window of 20 pair-words starting at LUT tick n0 - jb - 4, i.e. word LUT_OFF + n0 - jb - 4 of the row
                const float *w = st + (tap0 - 2 * jb0 - 8 * m);
                const float *cq = row + 4 + 4 * m;
                u64 Q0[4], Q1[4], Q2[4], Q3[4], Q4[4], cv[4];
                load4w(Q1, w + 8);  load4w(Q2, w + 16);  load4w(Q3, w + 24);  load4w(Q4, w + 32);
                while (true) {
                    load4w(Q0, w);  load4c(cv, cq);
                    fma_step(acc, cv, Q0, Q1, Q2, Q3, Q4);
                    w -= 8;  cq += 4;
                    if (++m > m_hi) break;
                    load4w(Q4, w);  load4c(cv, cq);
                    fma_step(acc, cv, Q4, Q0, Q1, Q2, Q3);
                    w -= 8;  cq += 4;
                    if (++m > m_hi) break;
                    load4w(Q3, w);  load4c(cv, cq);
                    fma_step(acc, cv, Q3, Q4, Q0, Q1, Q2);
                    w -= 8;  cq += 4;
                    if (++m > m_hi) break;
                    load4w(Q2, w);  load4c(cv, cq);
                    fma_step(acc, cv, Q2, Q3, Q4, Q0, Q1);
                    w -= 8;  cq += 4;
                    if (++m > m_hi) break;
                    load4w(Q1, w);  load4c(cv, cq);
                    fma_step(acc, cv, Q1, Q2, Q3, Q4, Q0);
                    w -= 8;  cq += 4;
                    if (++m > m_hi) break;
                }
            }
        }
        __syncwarp();
        DBG_T(t2);
        DBG_ADD(1, t2 - t1);
        if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(empty0 + 8u * s) : "memory");
        if (h.z & FLAG_LAST) {
            // partial waveforms of the tile out; accumulators back to zero for the next tile
            const int nB_lo = (h.z >> 8) & 0xff, nB_hi = (h.z >> 16) & 0xff;
            const int d0 = 2 * (g * p.PG + pl);
            if (valid && blk >= nB_lo && blk <= nB_hi) {
                float lo[NO], hi[NO];
#pragma unroll
                for (int i = 0; i < NO; ++i) {
                    lo[i] = __uint_as_float((unsigned)(acc[i] & 0xffffffffull));
                    hi[i] = __uint_as_float((unsigned)(acc[i] >> 32));
                }
                if (d0 < WW) {
                    float2 *dst = (float2 *)(a.partial + ((size_t)h.w * WW + d0) * p.tile_ticks + n0);
#pragma unroll
                    for (int q = 0; q < NO / 2; ++q) dst[q] = make_float2(lo[2 * q], lo[2 * q + 1]);
                }
                if (d0 + 1 < WW) {
                    float2 *dst = (float2 *)(a.partial + ((size_t)h.w * WW + d0 + 1) * p.tile_ticks + n0);
#pragma unroll
                    for (int q = 0; q < NO / 2; ++q) dst[q] = make_float2(hi[2 * q], hi[2 * q + 1]);
                }
            }
#pragma unroll
            for (int i = 0; i < NO; ++i) acc[i] = 0ull;
        }
        if (++s == S) { s = 0; ph ^= 1u; }
        DBG_T(t3);
        DBG_ADD(2, t3 - t2);
    }
}

int response_stage_floats(const DevParams &p)
{
    return p.PG * p.RS * 2 + 4 + ((p.CJ + 3) & ~3);                  // LUT rows, row header, charge row
}
int response_stages(const DevParams &p, size_t smem_limit_per_cta)
{
    const size_t stage = (size_t)response_stage_floats(p) * 4;
    int s = (int)((smem_limit_per_cta - 256) / stage);
    return s > 4 ? 4 : s;
}

}  // namespace

int launch_current_splat(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n,
                         lartpc_signals_t *out, cudaStream_t st)
{
    (void)n;
    const DevParams &p = sim->dp;
    if (sim->n_tiles == 0) return LARTPC_OK;
    SplatArgs a;
    a.p = p;
    a.tpcs = sim->d_tpcs;
    a.tile_cp = sim->tile_cp;  a.tile_desc = sim->tile_desc;   // the tensor-core splat walks the sorted copies (below)
    a.pix_start = sim->pix_start;  a.pix_count = sim->pix_count;  a.pair_seg = sim->pair_seg;
    a.q_anode = dr->q_anode;  a.sigma_T = dr->sigma_T;  a.sigma_t = dr->sigma_t;
    a.u_s = dr->u_s; a.v_s = dr->v_s; a.u_e = dr->u_e; a.v_e = dr->v_e; a.T_s = dr->T_s; a.T_e = dr->T_e;
    a.a_lo = pm->a_lo; a.a_hi = pm->a_hi; a.b_lo = pm->b_lo; a.b_hi = pm->b_hi;
    a.jt0 = pm->jt0; a.jt1 = pm->jt1; a.n_samples = pm->n_samples;
    a.charge = out->charge;  a.tile_range = out->tile_range;
    a.fma_counter = sim->d_fma;
    a.rec = nullptr;  a.tile_list = nullptr;  a.work = nullptr;  a.n_tiles = 0;  a.tb_mask = sim->tb_mask;  a.cmask = sim->tc_cmask;
    if (p.tc_mode) {
        // per-(unit, bin) block masks: the tensor-core splat ORs in what every tile charges; the FFMA2 splat does not
        // keep them, every bin then counts as charged
        const size_t words = (size_t)((sim->n_tiles + TC_UNIT_TILES - 1) / TC_UNIT_TILES) * TC_CMASK_WORDS;
        LARTPC_CUDA_TRY(cudaMemsetAsync(sim->tc_cmask, splat_on_tc(p) ? 0 : 0xff, sizeof(int32_t) * words, st));
    }
    if (p.rnd_m > 0 && !splat_on_tc(p)) return LARTPC_ERR_UNSUPPORTED;
    if (splat_on_tc(p)) {
        // tensor-core splat (charge_tc.cuh); other bin counts use the FFMA2 splat below, which writes the same image
        static SmemCfg cfg_tc[6];
#define LARTPC_CT_ATTR(I, NBV, R, C) LARTPC_CUDA_TRY(ensure_dyn_smem(charge_lattice_tc_kernel<NBV, R, C>, cfg_tc[I], sim->device, CT_SMEM))
        LARTPC_CT_ATTR(0, 10, false, false);  LARTPC_CT_ATTR(1, 5, false, false);
        LARTPC_CT_ATTR(2, 10, true, false);   LARTPC_CT_ATTR(3, 5, true, false);
        LARTPC_CT_ATTR(4, 10, false, true);   LARTPC_CT_ATTR(5, 5, false, true);
#undef LARTPC_CT_ATTR
        if (n >= (1ll << 30) || sim->n_tiles >= INT32_MAX - 8 * (int64_t)sim->sm_count) return LARTPC_ERR_UNSUPPORTED;
        if (n > sim->seg_rec_cap) return LARTPC_ERR_ORDER;                // records are written with the plan (launch_seg_records)
        a.rec = sim->seg_rec;  a.work = sim->d_work;  a.n_tiles = (int)sim->n_tiles;
        a.tile_desc = sim->tile_desc_p;  a.tile_list = sim->tile_list_p;        // physical (sorted) tile order
        LARTPC_CUDA_TRY(cudaMemsetAsync(sim->d_work, 0, sizeof(int), st));
        const unsigned grid = (unsigned)std::min<int64_t>(sim->n_tiles, LARTPC_CT_CTAS * (int64_t)sim->sm_count);
        ++g_lartpc_launches;
        if (p.rnd_m > 0) {
            if (p.nb == 10) charge_lattice_tc_kernel<10, true, false><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
            else charge_lattice_tc_kernel<5, true, false><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
        } else if (sim->need_composite) {                              // some segment is beyond the largest single rule
            if (p.nb == 10) charge_lattice_tc_kernel<10, false, true><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
            else charge_lattice_tc_kernel<5, false, true><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
        } else {
            if (p.nb == 10) charge_lattice_tc_kernel<10, false, false><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
            else charge_lattice_tc_kernel<5, false, false><<<grid, CT_THREADS, CT_SMEM, st>>>(a);
        }
        LARTPC_CUDA_TRY(cudaGetLastError());
        return LARTPC_OK;
    }
    size_t smem = splat_smem_bytes(p);
    static SmemCfg cfg_splat;
    LARTPC_CUDA_TRY(ensure_dyn_smem(charge_lattice_kernel, cfg_splat, sim->device, smem));
    ++g_lartpc_launches;
    charge_lattice_kernel<<<(unsigned)sim->n_tiles, NT1, smem, st>>>(a);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}


// Truth association (truth.cuh): shares of the segments in every hit of a list sorted by (pixel, tick)
int launch_hit_truth(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, const lartpc_hits_t *hits,
                     int64_t n_hits, lartpc_truth_t *out, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    if (n_hits == 0) return LARTPC_OK;
    if (p.rnd_m > 0 || p.nb > 15 || n_hits >= INT32_MAX) return LARTPC_ERR_UNSUPPORTED;
    if (!sim->d_cum_lut) {
        // running sum of the response over LUT ticks, built once per sim from the table lartpc_sim_create was given
        const size_t elems = sim->lut_copy.size();
        float *raw = nullptr;
        LARTPC_CUDA_TRY(cudaMalloc(&raw, elems * sizeof(float)));
        cudaError_t e = cudaMalloc(&sim->d_cum_lut, elems * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpyAsync(raw, sim->lut_copy.data(), elems * sizeof(float), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) {
            const long long n_series = (long long)(elems / (size_t)p.K);
            ++g_lartpc_launches;
            cum_lut_kernel<<<div_up(n_series, 128), 128, 0, st>>>(raw, sim->d_cum_lut, n_series, p.K);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(raw);
        if (e != cudaSuccess) {
            if (sim->d_cum_lut) cudaFree(sim->d_cum_lut);
            sim->d_cum_lut = nullptr;
            lartpc_note_cuda_error(e, __FILE__, __LINE__);
            return LARTPC_ERR_CUDA;
        }
    }
    TruthArgs a;
    a.p = p;
    a.tpcs = sim->d_tpcs;
    a.pix_start = sim->pix_start;  a.pix_count = sim->pix_count;  a.pair_seg = sim->pair_seg;
    a.q_anode = dr->q_anode;  a.sigma_T = dr->sigma_T;  a.sigma_t = dr->sigma_t;
    a.u_s = dr->u_s; a.v_s = dr->v_s; a.u_e = dr->u_e; a.v_e = dr->v_e; a.T_s = dr->T_s; a.T_e = dr->T_e;
    a.a_lo = pm->a_lo; a.a_hi = pm->a_hi; a.b_lo = pm->b_lo; a.b_hi = pm->b_hi;
    a.jt0 = pm->jt0; a.jt1 = pm->jt1; a.n_samples = pm->n_samples;
    a.cum_lut = sim->d_cum_lut;
    a.hit_pixel = hits->hit_pixel;  a.hit_tick = hits->hit_tick;
    a.n_hits = n_hits;  a.k_max = out->k_max;
    a.out_seg = out->seg;  a.out_frac = out->frac;  a.out_q = out->q_signal;  a.out_n = out->n_contrib;
    ++g_lartpc_launches;
    hit_truth_kernel<<<(unsigned)n_hits, TR_THREADS, 0, st>>>(a);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// per-segment records of the tensor-core splat, written once per plan of the whole input (launch_plan with tpc_lo = 0);
// sets d_counters[CNT_COMPOSITE] when some segment wants composite node rules
int launch_seg_records(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    if (!splat_on_tc(p) || n <= 0) return LARTPC_OK;
    if (n >= (1ll << 30)) return LARTPC_ERR_UNSUPPORTED;
    if (n > sim->seg_rec_cap) {
        if (sim->seg_rec) cudaFree(sim->seg_rec);
        sim->seg_rec = nullptr;  sim->seg_rec_cap = 0;
        LARTPC_CUDA_TRY(cudaMalloc(&sim->seg_rec, sizeof(SegRec) * (size_t)(n + n / 8 + 1024)));
        sim->seg_rec_cap = n + n / 8 + 1024;
    }
    ++g_lartpc_launches;
    seg_record_kernel<<<div_up(n, 256), 256, 0, st>>>(p, n, dr->q_anode, dr->sigma_T, dr->sigma_t, dr->u_s, dr->v_s,
                                                     dr->u_e, dr->v_e, dr->T_s, dr->T_e, pm->a_lo, pm->a_hi, pm->b_lo,
                                                     pm->b_hi, pm->jt0, pm->jt1, pm->n_samples, (SegRec *)sim->seg_rec,
                                                     sim->d_counters + CNT_COMPOSITE);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// two CTAs per SM: each may use half of the SM's shared memory minus the 1 KB the system reserves per CTA
static size_t response_smem_budget() { return (size_t)(228 * 1024) / 2 - 1024; }

int launch_current_response(lartpc_sim *sim, lartpc_signals_t *out, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    if (sim->n_tiles == 0) return LARTPC_OK;
    ResponseArgs a;
    a.p = p;
    a.lut = sim->d_lut;
    a.charge = out->charge;
    a.partial = out->partial;
    a.work = sim->d_work;
    const int64_t n_work = sim->n_tiles * p.n_groups;
    if (n_work >= INT32_MAX) return LARTPC_ERR_UNSUPPORTED;
    a.n_work = (int)n_work;
    a.stage_floats = response_stage_floats(p);
    a.lut_floats = p.PG * p.RS * 2;
    a.n_stages = response_stages(p, response_smem_budget());
    memcpy(a.blk_of_slot, sim->blk_of_slot, sizeof(a.blk_of_slot));
    a.end_row = sim->d_end_row;
    if (a.n_stages < 2) return LARTPC_ERR_UNSUPPORTED;
    size_t smem = (size_t)a.n_stages * a.stage_floats * 4 + 2 * (size_t)a.n_stages * sizeof(u64) + 64;   // + pair group per stage
    static SmemCfg cfg_resp;
    LARTPC_CUDA_TRY(ensure_dyn_smem(response_kernel, cfg_resp, sim->device, smem));
    LARTPC_CUDA_TRY(cudaMemsetAsync(sim->d_work, 0, sizeof(int), st));
    const int grid = (int)std::min<int64_t>(n_work, 2 * (int64_t)sim->sm_count);
    ++g_lartpc_launches;
    response_kernel<<<grid, NT2, smem, st>>>(a);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

#ifdef LARTPC_DEBUG_CLOCKS
extern "C" int lartpc_debug_clocks(unsigned long long out[32], int reset)
{
    cudaMemcpyFromSymbol(out, g_ct_dbg, sizeof(unsigned long long) * 8);   // charge lattice: thread 0's cycles per phase
    cudaMemcpyFromSymbol(out + 24, g_ct_dbg, sizeof(unsigned long long) * 8, sizeof(unsigned long long) * 8);
    cudaMemcpyFromSymbol(out + 8, rtc::g_rtc_dbg, sizeof(unsigned long long) * 16);
    if (reset) {
        unsigned long long z[16] = {0};
        cudaMemcpyToSymbol(g_ct_dbg, z, sizeof(unsigned long long) * 8);
        cudaMemcpyToSymbol(g_ct_dbg, z, sizeof(unsigned long long) * 8, sizeof(unsigned long long) * 8);
        cudaMemcpyToSymbol(rtc::g_rtc_dbg, z, sizeof(z));
    }
    return 0;
}
#endif

// shared-memory needs for a parameter set (used by lartpc_sim_create to pick the tile geometry)
size_t lartpc_splat_smem(const DevParams &p) { return splat_smem_bytes(p); }
size_t lartpc_response_smem(const DevParams &p)
{
    return 2 * (size_t)response_stage_floats(p) * 4 + 64;           // at least two stages must fit
}

// =====================================================================================================
// Tensor-core response: launcher and the LUT operand images
// =====================================================================================================
int launch_current_response_tc(lartpc_sim *sim, lartpc_signals_t *out, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    if (sim->n_tiles == 0) return LARTPC_OK;
    if (p.Jc != rtc::JC || !sim->d_lut_tc || 32 + p.NBW > rtc::ACC_COL) return LARTPC_ERR_UNSUPPORTED;
    constexpr bool PAIR = TC_CTA_PAIR;
    rtc::Args a;
    a.A = (const __half *)out->charge;
    a.B = (const __half *)sim->d_lut_tc;
    a.partial = out->partial;
    a.tile_meta = out->tile_range;
    a.tb_mask = sim->tb_mask;
    a.cmask = sim->tc_cmask;
    static_assert(rtc::CMW == TC_CMASK_WORDS, "one layout of the per-bin block masks");
    if (sim->n_tiles >= INT32_MAX) return LARTPC_ERR_UNSUPPORTED;
    a.n_tiles = (int)sim->n_tiles;
    a.n_units = (int)((sim->n_tiles + TC_UNIT_TILES - 1) / TC_UNIT_TILES);
    a.NC = p.NB2;  a.WW = p.WW * p.nq;  a.NBW = p.NBW;  a.tile_ticks = p.tile_ticks;   // a row = (target, LUT piece)
    a.b_scale_log2 = p.b_scale_log2;
    a.K = p.KQ;  a.kappa = p.trunc_kappa;
    a.n_items = (long long)a.n_units * a.WW;
    if (a.n_items >= INT32_MAX) return LARTPC_ERR_UNSUPPORTED;
    a.work = sim->d_work;
    a.stats = sim->d_fma;
    LARTPC_CUDA_TRY(cudaMemsetAsync(sim->d_work, 0, sizeof(int), st));
    a.n_stages = rtc::n_stages(p.NBW, PAIR, (size_t)227 * 1024);
    if (a.n_stages < 2) return LARTPC_ERR_UNSUPPORTED;
    const size_t smem = rtc::smem_bytes(p.NBW, PAIR, a.n_stages);
    static SmemCfg cfg_rtc;
    LARTPC_CUDA_TRY(ensure_dyn_smem(rtc::response_tc_kernel<PAIR>, cfg_rtc, sim->device, smem));
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr[1];
    const int per = PAIR ? 2 : 1;
    int clusters = sim->sm_count / per;
    cfg.blockDim = dim3(rtc::THREADS, 1, 1);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = per;  attr[0].val.clusterDim.y = 1;  attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;  cfg.numAttrs = 1;
    if (PAIR) {
        // CTA pairs that can be resident at once (one CTA per SM, both SMs of a pair in one TPC)
        cfg.gridDim = dim3((unsigned)(clusters * per), 1, 1);
        int max_clusters = 0;
        if (cudaOccupancyMaxActiveClusters(&max_clusters, rtc::response_tc_kernel<PAIR>, &cfg) == cudaSuccess && max_clusters > 0)
            clusters = std::min(clusters, max_clusters);
        else cudaGetLastError();
    }
    clusters = (int)std::min<long long>(clusters, a.n_items);
    cfg.gridDim = dim3((unsigned)(clusters * per), 1, 1);
    ++g_lartpc_launches;
    LARTPC_CUDA_TRY(cudaLaunchKernelEx(&cfg, rtc::response_tc_kernel<PAIR>, a));
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// Bs[d, q][c][CTA of the pair][fp16 | fp8][rows x 32 bytes] with Bs[n'][jj] = R[c][d][KQ q + n' - jj] * 2^b_scale_log2 (0 outside piece q of the LUT): the fp16 image
// (rtc::b_image_offset) and the fp8 image of the cross terms (rtc::b8_image_offset), both in the canonical un-swizzled
// K-major layout.  Built once per sim on the host.
size_t lartpc_build_lut_tc(const DevParams &p, const float *lut_host, void **d_out)
{
    const int nb = p.nb, W = p.W, NBW = p.NBW, NB = W * nb;
    const int split = TC_CTA_PAIR ? 2 : 1, rows = NBW / split;          // rows of a generator one CTA of the pair holds
    const size_t half_elems = (size_t)NBW * 16, n = (size_t)p.WW * p.nq * p.NB2 * 2 * half_elems;
    const size_t cta_halfs = (size_t)rows * 16;                         // halfs of one precision part of one CTA's rows
    std::vector<__half> img(n);
    for (int dq = 0; dq < p.WW * p.nq; ++dq) {                         // row = (target d, LUT piece q): ticks [KQ q, KQ q + K)
        const int d = dq / p.nq, q = dq - d * p.nq, K = std::min(p.KQ, p.K - p.KQ * q);
        const int dyi = d / W, dxi = d - dyi * W;
        for (int cb = 0; cb < nb; ++cb)
            for (int ca = 0; ca < nb; ++ca) {
                const float *src = lut_host + ((size_t)(nb * dyi + cb) * NB + (nb * dxi + ca)) * p.K + (size_t)p.KQ * q;
                __half *bin_img = img.data() + ((size_t)dq * p.NB2 + (cb * nb + ca)) * 2 * half_elems;
                for (int nn = 0; nn < NBW; ++nn) {
                    // (target, bin) image: [CTA of the pair][fp16 part | fp8 part], each part the canonical K-major
                    // image of that CTA's rows
                    const int rk = nn / rows, nl = nn - rk * rows;
                    __half *hi = bin_img + (size_t)rk * 2 * cta_halfs;
                    unsigned char *f8 = (unsigned char *)(hi + cta_halfs);
                    for (int jj = 0; jj < 16; ++jj) {
                        const int k = nn - jj;
                        const float x = (k >= 0 && k < K) ? ldexpf(src[k], p.b_scale_log2) : 0.f;
                        const __half h = __float2half_rn(x);
                        hi[rtc::b_image_offset(nl, jj)] = h;
                        f8[rtc::b8_image_offset(nl, jj)] =
                            __nv_cvt_float_to_fp8(ldexpf(x, -rtc::SA_LOG2), __NV_SATFINITE, __NV_E4M3);
                        f8[rtc::b8_image_offset(nl, 16 + jj)] =
                            __nv_cvt_float_to_fp8(ldexpf(x - __half2float(h), rtc::SB_LOG2), __NV_SATFINITE, __NV_E4M3);
                    }
                }
            }
    }
    if (cudaMalloc(d_out, n * sizeof(__half)) != cudaSuccess) return 0;
    if (cudaMemcpy(*d_out, img.data(), n * sizeof(__half), cudaMemcpyHostToDevice) != cudaSuccess) return 0;
    return n * sizeof(__half);
}
