// S4  induced current, eqs. (3.7)-(3.9) P:L660-687 with the M-sum in expectation (D1).
//
// Decomposition: the paper's kernel gives one thread to every (segment, pixel, tick)
// and lets it sum N*M LUT look-ups.  By linearity of eq. (3.7) the same sum is
//     C[b][a][j]  = sum_seg sum_mu (Q_a/N) wx[a] wy[b] wt[j]          (charge per LUT cell, eq. 3.8)
//     I_p[n]      = sum_{a,b,j} C[b][a][j] * R[b - nb(iy-H)][a - nb(ix-H)][n - j]      (eq. 3.7)
// which needs ~50x fewer operations and shares the charge lattice between neighbouring segments.
// One CTA owns one charge tile = (charged pixel P, chunk of Jc arrival ticks):
//   phase 1  splat the tile's segments into C[nb*nb][Jc] in shared memory (register-tiled outer products
//            of per-sample erf-difference weights, no atomics);
//   phase 2  find the non-empty bins and their tick ranges;
//   phase 3  response: a thread keeps 16 output ticks of a PAIR of target pixels in registers (32 accumulators
//            as 16 packed f32x2) and slides a 24-tap window of the pair-interleaved LUT rows over the charge row:
//            128 FFMA2 (256 multiply-adds) per 4 LDS.128 of taps + 2 broadcast LDS.128 of charge.  The LUT rows of
//            the next non-empty bin arrive by cp.async.bulk (TMA engine, mbarrier completion) into the other half
//            of a double buffer while the current bin is being used;
//   phase 4  the tile's partial waveforms go to global memory; S5 sums them per pixel in a fixed order.
#include "common.cuh"

namespace {

constexpr int NT = 256;          // threads per CTA (two CTAs per SM)
constexpr int NO = 16;           // output ticks per response task
constexpr int LUT_OFF = 16;      // LUT tick k sits at word LUT_OFF + k of its zero-padded row
constexpr int SB = 64;           // samples per splat batch
constexpr int XS = 16;           // row length of the per-sample x / y weight tables (bins_per_pixel <= 15)
constexpr int SEGCAP = 32;       // segments staged per batch

struct CurrentArgs {
    DevParams p;
    const DevTpc *tpcs;
    const int32_t *tile_cp;
    const TileDesc *tile_desc;
    const int32_t *pix_start, *pix_count, *pair_seg;
    const float *q_anode, *sigma_T, *sigma_t;
    const double *u_s, *v_s, *u_e, *v_e, *T_s, *T_e;
    const int32_t *a_lo, *a_hi, *b_lo, *b_hi, *jt0, *jt1, *n_samples;
    const float *lut;
    float *partial;
    int32_t *tile_range;
    unsigned long long *fma_counter;   // multiply-adds of the response: non-zero cells x valid targets x K
    int CJ, NEP, NB2P;           // smem strides: charge row, erf row, wxy row
};

struct SegLocal {               // one staged segment, tile-relative
    float as, ae, bs, be, ts, te, isT, ist, q;
    int N, alo, ahi, blo, bhi, jlo, jhi, seg, zero_sigma;
};

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
__device__ __forceinline__ void load8w(u64 (&d)[8], const float *s)    // 8 pair-words = 64 bytes
{
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        ulonglong2 v = *(const ulonglong2 *)(s + 4 * q);
        d[2 * q] = v.x;  d[2 * q + 1] = v.y;
    }
}
__device__ __forceinline__ void load8c(u64 (&c)[8], const float *s)    // 8 charges, each duplicated into a pair
{
    float4 x = *(const float4 *)s, y = *(const float4 *)(s + 4);
    c[0] = pack2(x.x); c[1] = pack2(x.y); c[2] = pack2(x.z); c[3] = pack2(x.w);
    c[4] = pack2(y.x); c[5] = pack2(y.y); c[6] = pack2(y.z); c[7] = pack2(y.w);
}
// acc[i] += sum_jj c[jj] * w[i - jj + 8],  w = lo[0..7] ++ mid[0..7] ++ hi[0..7]  (i < 16, jj < 8)
__device__ __forceinline__ void fma_step(u64 (&acc)[NO], const u64 (&c)[8], const u64 (&lo)[8], const u64 (&mid)[8],
                                         const u64 (&hi)[8])
{
#pragma unroll
    for (int jj = 0; jj < 8; ++jj)
#pragma unroll
        for (int i = 0; i < NO; ++i) {
            const int m = i - jj + 8;
            ffma2(acc[i], c[jj], m < 8 ? lo[m] : (m < 16 ? mid[m - 8] : hi[m - 16]));
        }
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
// one thread: expect `bytes` on the barrier and start the global -> shared bulk copy
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, void *bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

__global__ void __launch_bounds__(NT, 2) induced_current_kernel(const CurrentArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NB2 = p.NB2, CJ = a.CJ, nb = p.nb, K = p.K, WW = p.WW, RS = p.RS;

    float *Csm = (float *)smem_raw;                                  // [NB2][CJ] charge per (bin, arrival tick)
    float *scratch = Csm + NB2 * CJ;                                 // splat scratch, later the LUT stage
    const int stage_floats = p.PG * RS * 2;                          // one LUT stage: PG pair rows of RS pair-words
    size_t scratch_floats = max((size_t)2 * stage_floats, (size_t)SB * (2 * XS + CJ));
    int *s_int = (int *)(scratch + scratch_floats);
    int *bin_jlo = s_int, *bin_jhi = s_int + NB2, *bin_list = s_int + 2 * NB2;
    int *s_misc = bin_list + NB2;                                    // [0] n bins, [1] tile jlo, [2] tile jhi
    u64 *mbar = (u64 *)(s_misc + 8);                                 // [2] "stage full" barriers
    SegLocal *segs = (SegLocal *)(mbar + 2);

    const int tile = blockIdx.x;
    const TileDesc td = a.tile_desc[tile];
    const int cp = a.tile_cp[tile];
    const DevTpc &tp = a.tpcs[td.tpc];
    const int A_t = td.px * nb, B_t = td.py * nb, J_t = td.chunk * p.Jc;
    const int lstart = a.pix_start[cp], lcount = a.pix_count[cp];

    for (int i = tid; i < NB2 * CJ / 4; i += NT) ((float4 *)Csm)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    if (tid == 0) {
        mbar_init(&mbar[0], 1);
        mbar_init(&mbar[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

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
                for (int mu = tid; mu < L.N; mu += NT) {
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
                for (int r = warp; r < nsb * runs; r += NT / 32) {
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
                for (int unit = tid; unit < units; unit += NT) {
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

    // ------------------------------------------------------------------ phase 2: non-empty bins
    int nz_cells = 0;
    for (int c = warp; c < NB2; c += NT / 32) {
        int lo = INT_MAX, hi = -1;
        for (int j = lane; j < CJ; j += 32)
            if (Csm[c * CJ + j] != 0.f) { lo = min(lo, j); hi = max(hi, j); ++nz_cells; }
        for (int d = 16; d; d >>= 1) {
            lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, d));
            hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, d));
        }
        if (lane == 0) { bin_jlo[c] = lo; bin_jhi[c] = hi; }
    }
    __syncthreads();
    if (warp == 0) {
        int nbins = 0, tlo = INT_MAX, thi = -1;
        for (int base = 0; base < NB2; base += 32) {
            const int c = base + lane;
            const bool f = c < NB2 && bin_jhi[c] >= 0;
            const unsigned bal = __ballot_sync(0xffffffffu, f);
            if (f) {
                bin_list[nbins + __popc(bal & ((1u << lane) - 1u))] = c;
                tlo = min(tlo, bin_jlo[c]);  thi = max(thi, bin_jhi[c]);
            }
            nbins += __popc(bal);
        }
        for (int d = 16; d; d >>= 1) {
            tlo = min(tlo, __shfl_xor_sync(0xffffffffu, tlo, d));
            thi = max(thi, __shfl_xor_sync(0xffffffffu, thi, d));
        }
        if (lane == 0) { s_misc[0] = nbins; s_misc[1] = tlo; s_misc[2] = thi; }
    }
    __syncthreads();
    const int nbins = s_misc[0], tjlo = s_misc[1], tjhi = s_misc[2];
    if (nbins == 0) {
        if (tid == 0 && blockIdx.y == 0) { a.tile_range[2 * tile] = 1; a.tile_range[2 * tile + 1] = 0; }
        return;
    }
    if (blockIdx.y == 0) {
        // multiply-adds the method needs here: non-zero cells x in-plane targets x K
        for (int d = 16; d; d >>= 1) nz_cells += __shfl_xor_sync(0xffffffffu, nz_cells, d);
        const int vx = min(td.px + p.H, tp.nx - 1) - max(td.px - p.H, 0) + 1;
        const int vy = min(td.py + p.H, tp.ny - 1) - max(td.py - p.H, 0) + 1;
        if (lane == 0 && nz_cells && vx > 0 && vy > 0)
            atomicAdd(a.fma_counter, (unsigned long long)nz_cells * (unsigned long long)(vx * vy * K));
    }

    // ------------------------------------------------------------------ phase 3: response
    // this CTA's pair group g = blockIdx.y: pairs [g PG, (g+1) PG); its LUT stage for bin c is one contiguous block
    const int g = blockIdx.y;
    const uint32_t stage_bytes = (uint32_t)stage_floats * 4u;
    const float *lut_g = a.lut + (size_t)g * stage_floats;
    const size_t lut_bin_stride = (size_t)p.NP * RS * 2;
    float *Rsm0 = scratch, *Rsm1 = scratch + stage_floats;
    if (tid == 0) {
        // the splat used this memory through the generic proxy; order those accesses before the bulk copies
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        bulk_load(Rsm0, lut_g + bin_list[0] * lut_bin_stride, stage_bytes, &mbar[0]);
        if (nbins > 1) bulk_load(Rsm1, lut_g + bin_list[1] * lut_bin_stride, stage_bytes, &mbar[1]);
    }
    const int nB_lo = tjlo >> 4, nB_hi = (tjhi + K - 1) >> 4;          // 16-tick output blocks, tile-relative
    const int blk = tid / p.PG, pl = tid - blk * p.PG;
    const bool t_ok = blk <= nB_hi - nB_lo;
    const int n0 = NO * (nB_lo + blk);
    u64 acc[NO];
#pragma unroll
    for (int i = 0; i < NO; ++i) acc[i] = 0ull;
    for (int bi = 0; bi < nbins; ++bi) {
        const int c = bin_list[bi];
        float *Rsm = (bi & 1) ? Rsm1 : Rsm0;
        mbar_wait(&mbar[bi & 1], (uint32_t)((bi >> 1) & 1));
        if (t_ok) {
            const int jlo_c = bin_jlo[c], jhi_c = bin_jhi[c];
            // groups of 8 charges whose taps k = n - j meet [0, K) for some of this task's outputs
            int jb = max(jlo_c & ~7, (n0 - K + 1) & ~7);
            const int jb_end = min(jhi_c & ~7, n0 + 8);
            if (jb <= jb_end) {
                const float *Crow = Csm + c * CJ;
                // window of 24 pair-words starting at LUT tick n0 - jb - 8, i.e. word n0 - jb + 8 of the row
                const float *w = Rsm + (pl * RS + (n0 - jb + LUT_OFF - 8)) * 2;
                u64 G0[8], G1[8], G2[8], cv[8];
                load8w(G1, w + 16);  load8w(G2, w + 32);
                while (true) {
                    load8w(G0, w);  load8c(cv, Crow + jb);
                    fma_step(acc, cv, G0, G1, G2);
                    jb += 8;  w -= 16;
                    if (jb > jb_end) break;
                    load8w(G2, w);  load8c(cv, Crow + jb);
                    fma_step(acc, cv, G2, G0, G1);
                    jb += 8;  w -= 16;
                    if (jb > jb_end) break;
                    load8w(G1, w);  load8c(cv, Crow + jb);
                    fma_step(acc, cv, G1, G2, G0);
                    jb += 8;  w -= 16;
                    if (jb > jb_end) break;
                }
            }
        }
        __syncthreads();                                             // every reader is done with this stage
        if (tid == 0 && bi + 2 < nbins) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            bulk_load(Rsm, lut_g + bin_list[bi + 2] * lut_bin_stride, stage_bytes, &mbar[bi & 1]);
        }
    }

    // ------------------------------------------------------------------ phase 4: partial waveforms out
    if (t_ok) {
        const int d0 = 2 * (g * p.PG + pl);
        float lo[NO], hi[NO];
#pragma unroll
        for (int i = 0; i < NO; ++i) {
            lo[i] = __uint_as_float((unsigned)(acc[i] & 0xffffffffull));
            hi[i] = __uint_as_float((unsigned)(acc[i] >> 32));
        }
        if (d0 < WW) {
            float4 *dst = (float4 *)(a.partial + ((size_t)tile * WW + d0) * p.tile_ticks + n0);
#pragma unroll
            for (int q = 0; q < NO / 4; ++q) dst[q] = make_float4(lo[4 * q], lo[4 * q + 1], lo[4 * q + 2], lo[4 * q + 3]);
        }
        if (d0 + 1 < WW) {
            float4 *dst = (float4 *)(a.partial + ((size_t)tile * WW + d0 + 1) * p.tile_ticks + n0);
#pragma unroll
            for (int q = 0; q < NO / 4; ++q) dst[q] = make_float4(hi[4 * q], hi[4 * q + 1], hi[4 * q + 2], hi[4 * q + 3]);
        }
    }
    if (tid == 0 && g == 0) { a.tile_range[2 * tile] = nB_lo; a.tile_range[2 * tile + 1] = nB_hi; }
}

size_t current_smem_bytes(const DevParams &p, int &CJ, int &NEP, int &NB2P)
{
    CJ = p.Jc;
    NEP = ((2 * (p.nb + 1) + p.Jc + 1) + 3) & ~3;
    NB2P = (p.NB2 + 3) & ~3;
    size_t scratch = (size_t)2 * p.PG * p.RS * 2;
    size_t splat = (size_t)SB * (2 * XS + CJ);
    if (splat > scratch) scratch = splat;
    size_t ints = 3 * (size_t)p.NB2 + 8 + 4;                      // bin tables, misc, two 64-bit mbarriers
    size_t bytes = ((size_t)p.NB2 * CJ + scratch) * 4 + ints * 4;
    bytes = (bytes + 15) & ~(size_t)15;
    return bytes + sizeof(SegLocal) * SEGCAP;
}

}  // namespace

int launch_current(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n,
                   lartpc_signals_t *out, cudaStream_t st)
{
    (void)n;
    const DevParams &p = sim->dp;
    if (sim->n_tiles == 0) return LARTPC_OK;
    CurrentArgs a;
    a.p = p;
    a.tpcs = sim->d_tpcs;
    a.tile_cp = sim->tile_cp;  a.tile_desc = sim->tile_desc;
    a.pix_start = sim->pix_start;  a.pix_count = sim->pix_count;  a.pair_seg = sim->pair_seg;
    a.q_anode = dr->q_anode;  a.sigma_T = dr->sigma_T;  a.sigma_t = dr->sigma_t;
    a.u_s = dr->u_s; a.v_s = dr->v_s; a.u_e = dr->u_e; a.v_e = dr->v_e; a.T_s = dr->T_s; a.T_e = dr->T_e;
    a.a_lo = pm->a_lo; a.a_hi = pm->a_hi; a.b_lo = pm->b_lo; a.b_hi = pm->b_hi;
    a.jt0 = pm->jt0; a.jt1 = pm->jt1; a.n_samples = pm->n_samples;
    a.lut = sim->d_lut;
    a.partial = out->partial;  a.tile_range = out->tile_range;
    a.fma_counter = sim->d_fma;
    size_t smem = current_smem_bytes(p, a.CJ, a.NEP, a.NB2P);
    static size_t configured = 0;
    if (smem > configured) {
        LARTPC_CUDA_TRY(cudaFuncSetAttribute(induced_current_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)smem));
        configured = smem;
    }
    dim3 grid((unsigned)sim->n_tiles, (unsigned)p.n_groups);
    ++g_lartpc_launches;
    induced_current_kernel<<<grid, NT, smem, st>>>(a);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// shared-memory need of the S4 kernel for a parameter set (used by lartpc_sim_create to pick Jc)
size_t lartpc_current_smem(const DevParams &p)
{
    int a, b, c;
    return current_smem_bytes(p, a, b, c);
}
int lartpc_current_threads() { return NT; }
