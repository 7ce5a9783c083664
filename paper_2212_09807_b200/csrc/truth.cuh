// Truth association of hits with segments (reading D26).  Included by stage_current.cu
// inside its anonymous namespace, after charge_tc.cuh (SegRec, stage_segment, erf_fast, the node-rule tables).
//
// The paper propagates truth through the light path only ("the true track segment id ... contributing to each
// ADC sample"); this is the charge-side analogue.  By eqs. (3.7)-(3.9) the current on a pixel is a sum over segments,
// I_p[n] = sum_s I_{p,s}[n].  At the sample tick n_h of hit h the CSA holds the charge integrated over ticks n0 .. n_h
// (n0: the tick after the pixel's previous sample, or a later periodic reset), so the share of segment s is
//     q_{h,s} = sum_{n = n0}^{n_h} I_{p,s}[n]
//             = sum over the LUT cells (bin c of a source pixel sigma in the W x W window around p, arrival tick j) of
//               C_s[c][j] * (S[c, d][min(n_h - j, K - 1)] - S[c, d][n0 - 1 - j]),      S[c, d][k] = sum_{k' <= k} R[c][d][k']
// with C_s the charge lattice of segment s alone (eq. 3.8) and d the place of p in sigma's window: the time sum of the
// response collapses into two look-ups of the LUT's running sum S, so a share costs one term per charged cell instead of
// K.  The main path never forms C_s -- it adds the segments of a tile before it applies the response, which is where
// its ~50x saving over the paper's kernel comes from -- so the truth pass rebuilds it per (hit, segment, source pixel)
// with the same weights (erf differences at the node-rule nodes or the N midpoints, float64 indicator decisions for
// sigma = 0): it is an optional second pass, as the paper's own full-truth option is.
//
// One CTA per hit.  The candidates are the segment lists the plan keeps per charged pixel (pair_seg), of the W x W source
// pixels around the hit's pixel; a segment whose readout ticks miss [n0, n_h] is skipped at once.  Per candidate the
// operand columns (nodes) are taken 64 at a time: phase 1, thread = (column, axis) writes the column's x / y bin weights
// to shared memory; phase 2, thread = (column, arrival tick) forms the tick weight and sums weight x S-difference over
// the bins of the source pixel (consecutive threads = consecutive ticks = consecutive LUT addresses).  Shares of one
// segment reached through several source pixels meet in a shared-memory table keyed by segment id; the k_max largest
// |q_{h,s}| go out with their fractions of the hit's total.

constexpr int TR_THREADS = 128;
constexpr int TR_COLS = 64;                 // operand columns per pass
constexpr int TR_TABLE = 2048;              // distinct segments per hit kept apart (beyond: lumped, counted)

struct TruthArgs {
    DevParams p;
    const DevTpc *tpcs;
    const int32_t *pix_start, *pix_count, *pair_seg;
    const float *q_anode, *sigma_T, *sigma_t;
    const double *u_s, *v_s, *u_e, *v_e, *T_s, *T_e;
    const int32_t *a_lo, *a_hi, *b_lo, *b_hi, *jt0, *jt1, *n_samples;
    const float *cum_lut;                   // S[cy][cx][k], [W nb][W nb][K]
    const int32_t *hit_pixel, *hit_tick;
    long long n_hits;
    int k_max;
    int32_t *out_seg;  float *out_frac;  float *out_q;  int32_t *out_n;
};

// the record seg_record_kernel writes, for one segment, from the S2 / S3 arrays
__device__ __forceinline__ SegRec truth_record(const TruthArgs &a, int i)
{
    const DevParams &p = a.p;
    const double inv_bin = 1.0 / p.bin, inv_dt = 1.0 / p.dt;
    SegRec r;
    r.ub_s = a.u_s[i] * inv_bin;  r.ub_e = a.u_e[i] * inv_bin;
    r.vb_s = a.v_s[i] * inv_bin;  r.vb_e = a.v_e[i] * inv_bin;
    r.tk_s = (a.T_s[i] - p.t_origin) * inv_dt;  r.tk_e = (a.T_e[i] - p.t_origin) * inv_dt;
    const float sT = a.sigma_T[i], st = a.sigma_t[i];
    const bool zero_sigma = !(sT > 0.0f) || !(st > 0.0f);
    r.isT = zero_sigma ? 0.f : (float)(p.bin * 0.70710678118654752440 / (double)sT);
    r.ist = zero_sigma ? 0.f : (float)(p.dt * 0.70710678118654752440 / (double)st);
    r.qa = a.q_anode[i];
    r.rho = 1.41421356f * fmaxf(fmaxf(fabsf((float)(r.ub_e - r.ub_s)), fabsf((float)(r.vb_e - r.vb_s))) * r.isT,
                                fabsf((float)(r.tk_e - r.tk_s)) * r.ist);
    r.N = a.n_samples[i];
    r.a_lo = a.a_lo[i]; r.a_hi = a.a_hi[i]; r.b_lo = a.b_lo[i]; r.b_hi = a.b_hi[i]; r.jt0 = a.jt0[i]; r.jt1 = a.jt1[i];
    r.flags = (int)((unsigned)i << 1) | (zero_sigma ? 1 : 0);
    return r;
}

// position along the segment and charge of operand column mu (charge_lattice_tc_kernel's column set-up, COMP form)
__device__ __forceinline__ void truth_column(const SegLocal &L, int mu, float &f, float &qw)
{
    f = ((float)mu + 0.5f) * (1.0f / (float)L.N);
    qw = L.q;
    if (L.rule >= 0) {
        if ((L.rule >> 16) == 0) {
            const float4 r = __ldg(&g_quad[(L.rule & 0xff) + mu]);
            f = r.x;
            qw = L.qa * (r.y - r.z * L.inv_n2 + r.w * L.inv_n4);
        } else {
            const unsigned rule_n = (unsigned)(L.rule >> 8) & 0xffu, pieces = (unsigned)(L.rule >> 16) + 1u;
            const unsigned pc = (unsigned)mu / rule_n;
            const int i = mu - (int)(pc * rule_n);
            const int s_p = (int)(pc * (unsigned)L.N / pieces), e_p = (int)((pc + 1u) * (unsigned)L.N / pieces);
            const float n_p = (float)(e_p - s_p), inv_n = 1.0f / (float)L.N, i2 = 1.0f / (n_p * n_p);
            const float4 r = __ldg(&g_quad[(L.rule & 0xff) + i]);
            f = ((float)s_p + r.x * n_p) * inv_n;
            qw = L.qa * (n_p * inv_n) * (r.y - r.z * i2 + r.w * i2 * i2);
        }
    }
}

__global__ void __launch_bounds__(TR_THREADS) hit_truth_kernel(const TruthArgs a)
{
    __shared__ float s_wx[TR_COLS][16], s_wy[TR_COLS][16];          // x / y bin weights of the columns of a pass
    __shared__ float s_pt[TR_COLS], s_q[TR_COLS];                   // arrival tick (relative) and charge of a column
    __shared__ int s_jj[TR_COLS];                                   // sigma = 0: the one arrival tick of a column (absolute), -1 none
    __shared__ int s_key[TR_TABLE];
    __shared__ float s_val[TR_TABLE];
    __shared__ double s_red[TR_THREADS / 32];
    __shared__ int s_hdr[8];                                        // tpc, ix, iy, n0, n_h, entries, -, -
    __shared__ float s_best[TR_THREADS / 32];
    __shared__ int s_besti[TR_THREADS / 32];
    __shared__ double s_other;
    __shared__ int s_cand[TR_THREADS], s_wn[TR_THREADS / 32];       // segments of a list pass whose current can reach the hit

    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long h = blockIdx.x;
    const int nb = p.nb, K = p.K, NBW = p.W * p.nb;
    DevParams p2 = p;                                               // staging without the 64-tick tile window, expectation form
    p2.Jc = 1 << 28;  p2.rnd_m = 0;

    for (int i = tid; i < TR_TABLE; i += TR_THREADS) { s_key[i] = -1;  s_val[i] = 0.f; }
    if (tid == 0) {
        const int pid = a.hit_pixel[h], n_h = a.hit_tick[h];
        int n0 = (h > 0 && a.hit_pixel[h - 1] == pid) ? a.hit_tick[h - 1] + 1 : 0;
        if (p.periodic > 0) {                                       // a periodic reset up to the crossing tick restarts the integral
            const int crossing = n_h - p.hold;
            const int r = crossing >= 0 ? (crossing / p.periodic) * p.periodic : 0;
            if (r >= 1 && r > n0) n0 = r;
        }
        int tpc = -1;
        for (int t = 0; t < p.n_tpcs; ++t) {
            const int rel = pid - a.tpcs[t].first_pixel_id;
            if (rel >= 0 && rel < a.tpcs[t].nx * a.tpcs[t].ny) { tpc = t;  s_hdr[1] = rel % a.tpcs[t].nx;  s_hdr[2] = rel / a.tpcs[t].nx;  break; }
        }
        s_hdr[0] = tpc;  s_hdr[3] = n0;  s_hdr[4] = n_h;  s_hdr[5] = 0;
        s_other = 0.0;
    }
    __syncthreads();
    const int tpc = s_hdr[0], ix = s_hdr[1], iy = s_hdr[2], n0 = s_hdr[3], n_h = s_hdr[4];

    if (tpc >= 0) {
        const DevTpc &t = a.tpcs[tpc];
        for (int ci = 0; ci < p.WW; ++ci) {
            const int dx = ci % p.W - p.H, dy = ci / p.W - p.H;
            const int sx = ix + dx, sy = iy + dy;                   // source pixel (may lie in the +-H margin outside the plane)
            const int cp = t.cp_base + (sy + p.H) * t.gw + (sx + p.H);
            const int lstart = a.pix_start[cp], lcount = a.pix_count[cp];
            // bin (al, bl) of the source pixel is seen by the hit's pixel through LUT column (al + nb (H - dx), ...): D5
            const int cx0 = nb * (p.H + dx), cy0 = nb * (p.H + dy);
            // the list holds every segment that ever charged the source pixel (~120 over a full spill); the threads first
            // pick, 128 entries at a time and in list order, those whose current can reach [n0, n_h] at all (two loads each:
            // a record costs nineteen), then the CTA takes the picked ones one by one
            for (int base = 0; base < lcount; base += TR_THREADS) {
            int n_cand;
            {
                const int li = base + tid;
                bool keep = false;
                int sc = -1;
                if (li < lcount) {
                    sc = a.pair_seg[lstart + li];
                    const int lo = max(a.jt0[sc], 0), hi = min(a.jt1[sc], p.j_max);
                    keep = lo <= hi && hi + K - 1 >= n0 && lo <= n_h;
                }
                const unsigned bal = __ballot_sync(0xffffffffu, keep);
                __syncthreads();                                    // (the last pass is done with s_cand)
                if (lane == 0) s_wn[warp] = __popc(bal);
                __syncthreads();
                int off = 0;
                n_cand = 0;
                for (int w = 0; w < TR_THREADS / 32; ++w) { if (w < warp) off += s_wn[w];  n_cand += s_wn[w]; }
                if (keep) s_cand[off + __popc(bal & ((1u << lane) - 1u))] = sc;
                __syncthreads();
            }
            for (int qi = 0; qi < n_cand; ++qi) {
                const int s = s_cand[qi];
                const SegRec rec = truth_record(a, s);
                const int J_t = max(rec.jt0, 0) & ~3;
                SegLocal L;
                const int nq = stage_segment<true>(p2, rec, s, nb, sx * nb, sy * nb, J_t, L);
                if (nq == 0) continue;                              // CTA-uniform (every thread stages the same record)
                if (J_t + L.jhi + K - 1 < n0 || J_t + L.jlo > n_h) continue;      // its current misses the window
                const int nj = L.jhi - L.jlo + 1;
                float acc = 0.f;
                for (int c0 = 0; c0 < nq; c0 += TR_COLS) {
                    const int ncol = min(TR_COLS, nq - c0);
                    __syncthreads();
                    {   // ---- phase 1: thread = (column, axis)
                        const int col = tid >> 1, axis = tid & 1;
                        if (col < ncol) {
                            const int mu = c0 + col;
                            float f, qw;
                            truth_column(L, mu, f, qw);
                            float *w = axis ? s_wy[col] : s_wx[col];
                            const int lo = axis ? L.blo : L.alo, hi = axis ? L.bhi : L.ahi;
                            if (L.zero_sigma) {
                                // the bin / tick is an integer decision taken in float64 in the oracle's order
                                const double fd = xdiv(xadd((double)mu, 0.5), (double)L.N);
                                const double ps = axis ? a.v_s[s] : a.u_s[s], pe = axis ? a.v_e[s] : a.u_e[s];
                                const double pos = xadd(ps, xmul(xsub(pe, ps), fd));
                                const long long xb = (long long)floor(xdiv(pos, p.bin)) - (long long)(axis ? sy : sx) * nb;
                                for (int i = 0; i < nb; ++i) w[i] = (i == xb) ? 1.f : 0.f;
                                if (axis == 0) {
                                    const double Ts = a.T_s[s], Te = a.T_e[s];
                                    const double TT = xadd(Ts, xmul(xsub(Te, Ts), fd));
                                    const long long j = (long long)floor(xdiv(xsub(TT, p.t_origin), p.dt));
                                    s_jj[col] = (j >= 0 && j <= p.j_max) ? (int)j : -1;
                                    s_q[col] = qw;
                                }
                            } else {
                                const float ps = axis ? L.bs : L.as, pe = axis ? L.be : L.ae;
                                const float pos = fmaf(pe - ps, f, ps);
                                float e0 = erf_fast((0.f - pos) * L.isT);
                                for (int i = 0; i < nb; ++i) {
                                    const float e1 = erf_fast(((float)(i + 1) - pos) * L.isT);
                                    w[i] = (i >= lo && i <= hi) ? 0.5f * (e1 - e0) : 0.f;
                                    e0 = e1;
                                }
                                if (axis == 0) { s_pt[col] = fmaf(L.te - L.ts, f, L.ts);  s_q[col] = 0.5f * qw; }
                            }
                        }
                    }
                    __syncthreads();
                    // ---- phase 2: thread = (column, arrival tick)
                    for (int item = tid; item < ncol * nj; item += TR_THREADS) {
                        const int col = item / nj, j = L.jlo + (item - col * nj), j_abs = J_t + j;
                        const int k1 = min(n_h - j_abs, K - 1), k0 = n0 - 1 - j_abs;
                        if (k1 < 0 || k0 >= K - 1) continue;          // the response of this tick lies outside the window
                        float wt;
                        if (L.zero_sigma) wt = (j_abs == s_jj[col]) ? s_q[col] : 0.f;
                        else {
                            const float pt = s_pt[col];
                            wt = s_q[col] * (erf_fast(((float)(j + 1) - pt) * L.ist) - erf_fast(((float)j - pt) * L.ist));
                        }
                        if (wt == 0.f) continue;
                        float sum = 0.f;
                        for (int b = L.blo; b <= L.bhi; ++b) {
                            const float wy = s_wy[col][b];
                            if (wy == 0.f) continue;
                            const float *S = a.cum_lut + ((size_t)(cy0 + b) * NBW + cx0) * K;
                            float row = 0.f;
                            for (int c = L.alo; c <= L.ahi; ++c) {
                                const float *Sc = S + (size_t)c * K;
                                const float v = __ldg(Sc + k1) - (k0 >= 0 ? __ldg(Sc + k0) : 0.f);
                                row = fmaf(s_wx[col][c], v, row);
                            }
                            sum = fmaf(wy, row, sum);
                        }
                        acc = fmaf(wt, sum, acc);
                    }
                }
                // ---- share of (segment, source pixel): block sum, then into the table
                double v = (double)acc;
                for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
                __syncthreads();
                if (lane == 0) s_red[warp] = v;
                __syncthreads();
                if (tid == 0) {
                    double share = 0.0;
                    for (int w = 0; w < TR_THREADS / 32; ++w) share += s_red[w];
                    if (share != 0.0) {
                        unsigned slot = ((unsigned)s * 2654435761u) >> 21;      // 11 bits
                        int probes = 0;
                        while (s_key[slot] != s && s_key[slot] != -1 && probes < TR_TABLE) { slot = (slot + 1) & (TR_TABLE - 1);  ++probes; }
                        if (s_key[slot] == s) s_val[slot] += (float)share;
                        else if (s_key[slot] == -1 && s_hdr[5] < TR_TABLE - 1) { s_key[slot] = s;  s_val[slot] = (float)share;  ++s_hdr[5]; }
                        else s_other += share;
                    }
                }
            }
            }
        }
    }
    __syncthreads();
    // ---- totals and the k_max largest shares
    double tot = 0.0;
    int cnt = 0;
    for (int i = tid; i < TR_TABLE; i += TR_THREADS)
        if (s_key[i] >= 0) { tot += (double)s_val[i];  cnt += s_val[i] != 0.f; }
    for (int d = 16; d; d >>= 1) { tot += __shfl_xor_sync(0xffffffffu, tot, d);  cnt += __shfl_xor_sync(0xffffffffu, cnt, d); }
    __shared__ int s_cnt[TR_THREADS / 32];
    if (lane == 0) { s_red[warp] = tot;  s_cnt[warp] = cnt; }
    __syncthreads();
    tot = s_other;  cnt = 0;
    for (int w = 0; w < TR_THREADS / 32; ++w) { tot += s_red[w];  cnt += s_cnt[w]; }
    const float inv = tot != 0.0 ? (float)(1.0 / tot) : 0.f;
    if (tid == 0) { a.out_q[h] = (float)tot;  a.out_n[h] = cnt + (s_other != 0.0 ? 1 : 0); }
    for (int k = 0; k < a.k_max; ++k) {
        // largest |share| still in the table; ties go to the lower segment id
        float best = -1.f;  int bi = -1;
        for (int i = tid; i < TR_TABLE; i += TR_THREADS) {
            if (s_key[i] < 0) continue;
            const float m = fabsf(s_val[i]);
            if (m > best || (m == best && bi >= 0 && s_key[i] < s_key[bi])) { best = m;  bi = i; }
        }
        for (int d = 16; d; d >>= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, d);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, d);
            if (oi >= 0 && (ob > best || (ob == best && (bi < 0 || s_key[oi] < s_key[bi])))) { best = ob;  bi = oi; }
        }
        __syncthreads();
        if (lane == 0) { s_best[warp] = best;  s_besti[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            best = -1.f;  bi = -1;
            for (int w = 0; w < TR_THREADS / 32; ++w) {
                const int oi = s_besti[w];
                if (oi >= 0 && (s_best[w] > best || (s_best[w] == best && (bi < 0 || s_key[oi] < s_key[bi])))) { best = s_best[w];  bi = oi; }
            }
            if (bi >= 0 && best > 0.f) {
                a.out_seg[h * a.k_max + k] = s_key[bi];
                a.out_frac[h * a.k_max + k] = s_val[bi] * inv;
                s_key[bi] = -2;                                     // taken
            } else {
                a.out_seg[h * a.k_max + k] = -1;
                a.out_frac[h * a.k_max + k] = 0.f;
            }
        }
        __syncthreads();
    }
}

// S[cy][cx][k] = sum_{k' <= k} R[cy][cx][k'], summed in float64: one thread per (cy, cx) series
__global__ void __launch_bounds__(128) cum_lut_kernel(const float *__restrict__ lut, float *__restrict__ cum, long long n_series, int K)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_series) return;
    double s = 0.0;
    for (int k = 0; k < K; ++k) { s += (double)lut[i * K + k];  cum[i * K + k] = (float)s; }
}
