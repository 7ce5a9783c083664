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
//   phase 3  response: every thread keeps TPT x 8 output ticks of one of the W*W target pixels in registers
//            and slides a 16-tap LUT window from shared memory over the charge row (64 FMA per 4 LDS.128);
//            the LUT rows of the current bin are staged from L2 into shared memory;
//   phase 4  the tile's partial waveforms go to global memory; S5 sums them per pixel in a fixed order.
#include "common.cuh"

namespace {

constexpr int NT = 512;          // threads per CTA
constexpr int TPT = 2;           // output tasks (target pixel x 8-tick block) per thread
constexpr int SB = 32;           // samples per splat batch
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

__device__ __forceinline__ void load8(float (&d)[8], const float *s)
{
    float4 x = *(const float4 *)s, y = *(const float4 *)(s + 4);
    d[0] = x.x; d[1] = x.y; d[2] = x.z; d[3] = x.w; d[4] = y.x; d[5] = y.y; d[6] = y.z; d[7] = y.w;
}

// acc[i] += sum_jj c[jj] * w[i - jj + 7],  w = lo[0..7] ++ hi[0..7]
__device__ __forceinline__ void fma_block(float (&acc)[8], const float (&c)[8], const float (&lo)[8],
                                          const float (&hi)[8])
{
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int jj = 0; jj < 8; ++jj) {
            const int m = i - jj + 7;
            acc[i] = fmaf(c[jj], m < 8 ? lo[m] : hi[m - 8], acc[i]);
        }
}

__global__ void __launch_bounds__(NT, 1) induced_current_kernel(const CurrentArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NB2 = p.NB2, CJ = a.CJ, nb = p.nb, K = p.K, WW = p.WW, RS = p.RS;

    float *Csm = (float *)smem_raw;                                  // [NB2][CJ] charge per (bin, arrival tick)
    float *scratch = Csm + NB2 * CJ;                                 // splat scratch, later the LUT stage
    size_t scratch_floats = max((size_t)WW * RS, (size_t)SB * (a.NEP + a.NB2P + CJ));
    int *s_int = (int *)(scratch + scratch_floats);
    int *bin_jlo = s_int, *bin_jhi = s_int + NB2, *bin_list = s_int + 2 * NB2, *valid_list = s_int + 3 * NB2;
    int *s_misc = valid_list + WW;                                   // [0] n bins, [1] tile jlo, [2] tile jhi, [3] nvalid
    SegLocal *segs = (SegLocal *)(s_misc + 8);

    const int tile = blockIdx.x;
    const TileDesc td = a.tile_desc[tile];
    const int cp = a.tile_cp[tile];
    const DevTpc &tp = a.tpcs[td.tpc];
    const int A_t = td.px * nb, B_t = td.py * nb, J_t = td.chunk * p.Jc;
    const int lstart = a.pix_start[cp], lcount = a.pix_count[cp];

    for (int i = tid; i < NB2 * CJ / 4; i += NT) ((float4 *)Csm)[i] = make_float4(0.f, 0.f, 0.f, 0.f);

    // ------------------------------------------------------------------ phase 1: splat
    float *erfv = scratch, *wxy = scratch + SB * a.NEP, *wt = wxy + SB * a.NB2P;
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
            const int ncell = na * nbb, ncell4 = (ncell + 3) >> 2, nj4 = (nj + 3) >> 2;
            const int nex = na + 1, ney = nbb + 1, ne = nex + ney + nj + 1;
            const float invN = 1.0f / (float)L.N;
            for (int mu0 = 0; mu0 < L.N; mu0 += SB) {
                const int nsb = min(SB, L.N - mu0);
                // (A) erf at every bin / tick edge of the segment's box for each sample of the batch
                for (int idx = tid; idx < nsb * ne; idx += NT) {
                    const int ml = idx / ne, e = idx - ml * ne;
                    const float f = ((float)(mu0 + ml) + 0.5f) * invN;
                    float arg;
                    if (e < nex)            arg = ((float)(L.alo + e) - fmaf(L.ae - L.as, f, L.as)) * L.isT;
                    else if (e < nex + ney) arg = ((float)(L.blo + e - nex) - fmaf(L.be - L.bs, f, L.bs)) * L.isT;
                    else                    arg = ((float)(L.jlo + e - nex - ney) - fmaf(L.te - L.ts, f, L.ts)) * L.ist;
                    erfv[ml * a.NEP + e] = erff(arg);
                }
                __syncthreads();
                // (B) cell weights: wxy = q (Phi_y[b+1]-Phi_y[b]) (Phi_x[a+1]-Phi_x[a]), wt = Phi_t[j+1]-Phi_t[j]
                for (int idx = tid; idx < nsb * (ncell4 * 4); idx += NT) {
                    const int ml = idx / (ncell4 * 4), c = idx - ml * (ncell4 * 4);
                    float w = 0.f;
                    if (c < ncell) {
                        const int b = c / na, aa = c - b * na;
                        const float *E = erfv + ml * a.NEP;
                        w = 0.25f * L.q * (E[nex + b + 1] - E[nex + b]) * (E[aa + 1] - E[aa]);
                    }
                    wxy[ml * a.NB2P + c] = w;
                }
                for (int idx = tid; idx < nsb * (nj4 * 4); idx += NT) {
                    const int ml = idx / (nj4 * 4), jj = idx - ml * (nj4 * 4);
                    const float *E = erfv + ml * a.NEP + nex + ney;
                    wt[ml * CJ + jj] = jj < nj ? 0.5f * (E[jj + 1] - E[jj]) : 0.f;
                }
                __syncthreads();
                // (C) accumulate 4 cells x 4 ticks per thread over the batch
                for (int unit = tid; unit < ncell4 * nj4; unit += NT) {
                    const int cq = unit / nj4, jq = unit - cq * nj4;
                    float acc[4][4];
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int k = 0; k < 4; ++k) acc[i][k] = 0.f;
                    const float *pw = wxy + cq * 4, *pt = wt + jq * 4;
                    for (int ml = 0; ml < nsb; ++ml) {
                        const float4 w4 = *(const float4 *)(pw + ml * a.NB2P);
                        const float4 t4 = *(const float4 *)(pt + ml * CJ);
                        const float wv[4] = {w4.x, w4.y, w4.z, w4.w}, tv[4] = {t4.x, t4.y, t4.z, t4.w};
#pragma unroll
                        for (int i = 0; i < 4; ++i)
#pragma unroll
                            for (int k = 0; k < 4; ++k) acc[i][k] = fmaf(wv[i], tv[k], acc[i][k]);
                    }
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int c = cq * 4 + i;
                        if (c < ncell) {
                            const int b = c / na, aa = c - b * na;
                            float *row = Csm + ((L.blo + b) * nb + (L.alo + aa)) * CJ + L.jlo + jq * 4;
#pragma unroll
                            for (int k = 0; k < 4; ++k)
                                if (jq * 4 + k < nj) row[k] += acc[i][k];
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
        int nvalid = 0;                       // targets inside the plane: ix = px + H - dxi, iy = py + H - dyi
        for (int base = 0; base < WW; base += 32) {
            const int d = base + lane;
            bool f = false;
            if (d < WW) {
                const int dyi = d / p.W, dxi = d - dyi * p.W;
                const int ix = td.px + p.H - dxi, iy = td.py + p.H - dyi;
                f = ix >= 0 && ix < tp.nx && iy >= 0 && iy < tp.ny;
            }
            const unsigned bal = __ballot_sync(0xffffffffu, f);
            if (f) valid_list[nvalid + __popc(bal & ((1u << lane) - 1u))] = d;
            nvalid += __popc(bal);
        }
        if (lane == 0) { s_misc[0] = nbins; s_misc[1] = tlo; s_misc[2] = thi; s_misc[3] = nvalid; }
    }
    __syncthreads();
    const int nbins = s_misc[0], tjlo = s_misc[1], tjhi = s_misc[2], nvalid = s_misc[3];
    if (blockIdx.y == 0) {
        for (int d = 16; d; d >>= 1) nz_cells += __shfl_xor_sync(0xffffffffu, nz_cells, d);
        if (lane == 0 && nz_cells)
            atomicAdd(a.fma_counter, (unsigned long long)nz_cells * (unsigned long long)(nvalid * K));
    }
    if (nbins == 0 || nvalid == 0) {
        if (tid == 0 && blockIdx.y == 0) { a.tile_range[2 * tile] = 1; a.tile_range[2 * tile + 1] = 0; }
        return;
    }

    // ------------------------------------------------------------------ phase 3: response
    const int nB_lo = tjlo >> 3, nB_hi = (tjhi + K - 1) >> 3;
    const int ntasks = nvalid * (nB_hi - nB_lo + 1);
    int t_delta[TPT], t_nB[TPT];
    bool t_ok[TPT];
    float acc[TPT][8];
#pragma unroll
    for (int s = 0; s < TPT; ++s) {
        const int task = (blockIdx.y * TPT + s) * NT + tid;
        t_ok[s] = task < ntasks;
        const int nBi = t_ok[s] ? task / nvalid : 0;
        t_delta[s] = valid_list[t_ok[s] ? task - nBi * nvalid : 0];
        t_nB[s] = nB_lo + nBi;
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[s][i] = 0.f;
    }
    float *Rsm = scratch;                                            // [WW][RS]: word 7 + k holds LUT tick k
    for (int bi = 0; bi < nbins; ++bi) {
        const int c = bin_list[bi];
        __syncthreads();                                             // previous bin's readers are done
        const float4 *src = (const float4 *)(a.lut + (size_t)c * WW * RS);
        for (int i = tid; i < WW * RS / 4; i += NT) ((float4 *)Rsm)[i] = __ldg(src + i);
        __syncthreads();
        const int jlo_c = bin_jlo[c], jhi_c = bin_jhi[c];
        const float *Crow = Csm + c * CJ;
#pragma unroll
        for (int s = 0; s < TPT; ++s) {
            if (!t_ok[s]) continue;
            const int n8 = 8 * t_nB[s];
            // j blocks whose 8x8 (n, j) square meets the band 0 <= n - j < K
            int jb = max(jlo_c & ~7, ((n8 - (K + 6) + 7) >> 3) << 3);
            const int jb_end = min(jhi_c & ~7, n8);
            if (jb > jb_end) continue;
            const float *rowp = Rsm + t_delta[s] * RS;
            int base = n8 - jb;                                      // window words [base, base+16)
            float A[8], B[8], cv[8];
            load8(B, rowp + base + 8);
            while (true) {
                load8(A, rowp + base);  load8(cv, Crow + jb);
                fma_block(acc[s], cv, A, B);
                jb += 8;  base -= 8;
                if (jb > jb_end) break;
                load8(B, rowp + base);  load8(cv, Crow + jb);
                fma_block(acc[s], cv, B, A);
                jb += 8;  base -= 8;
                if (jb > jb_end) break;
            }
        }
    }

    // ------------------------------------------------------------------ phase 4: partial waveforms out
#pragma unroll
    for (int s = 0; s < TPT; ++s) {
        if (!t_ok[s]) continue;
        float *dst = a.partial + ((size_t)tile * WW + t_delta[s]) * p.tile_ticks + 8 * t_nB[s];
        *(float4 *)dst = make_float4(acc[s][0], acc[s][1], acc[s][2], acc[s][3]);
        *(float4 *)(dst + 4) = make_float4(acc[s][4], acc[s][5], acc[s][6], acc[s][7]);
    }
    if (tid == 0 && blockIdx.y == 0) { a.tile_range[2 * tile] = nB_lo; a.tile_range[2 * tile + 1] = nB_hi; }
}

size_t current_smem_bytes(const DevParams &p, int &CJ, int &NEP, int &NB2P)
{
    CJ = p.Jc;
    NEP = ((2 * (p.nb + 1) + p.Jc + 1) + 3) & ~3;
    NB2P = (p.NB2 + 3) & ~3;
    size_t scratch = (size_t)p.WW * p.RS;
    size_t splat = (size_t)SB * (NEP + NB2P + CJ);
    if (splat > scratch) scratch = splat;
    size_t ints = 3 * (size_t)p.NB2 + p.WW + 8;
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
int lartpc_current_tasks_per_group() { return NT * TPT; }
