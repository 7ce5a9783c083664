// S4 charge lattice on the tensor cores (included by stage_current.cu inside its anonymous namespace, after SplatArgs
// and SegLocal).  Eq. (3.8) in expectation, reading D1:
//     C[b][a][j] = sum_seg sum_mu (Q_a / N) wx_mu[a] wy_mu[b] wt_mu[j]
// is, per tile, the matrix product  D[m = b nb + a][j] = sum_s WXY[m][s] WT[j][s]  over the samples s of every segment
// that crosses the tile: M = 128 cell rows (nb^2 = 100 used), N = 64 arrival ticks, K = samples.  Persistent CTAs of
// 128 threads (four per SM) take tiles from an atomic cursor; 64 samples per batch: warps 0-1 build the WXY operand of
// their sample (11 + 11 erf, 100 products), warps 2-3 the WT operand (up to 65 erf), both split hi + lo in fp16 and
// stored MN-major (a thread writes 16-byte runs of cells / ticks of its own sample column: conflict-free STS.128) in the
// canonical un-swizzled UMMA layout; thread 0 then issues 3 x ceil(samples / 16) tcgen05.mma (hi hi + hi lo + lo hi)
// into a 64-column TMEM accumulator (allocated once per CTA).  When the last segment is in, every thread reads its cell
// row from TMEM, the tile's scale exponent is agreed on, and the row goes out as the operand image the tensor-core
// response reads (rtc::store_a_block16).
// What a tile needs from global memory -- its descriptor, the segment ids of its pixel, one 96-byte record per segment
// (seg_record_kernel) -- is fetched by warp 0 with cp.async while the tiles before it are computed: descriptor two
// tiles ahead, ids one tile ahead, records during the previous tile; nothing on that chain is waited for.
// sigma = 0 segments take the float64 indicator path of the oracle (one-hot weights), as in charge_lattice_kernel.

constexpr int CT_THREADS = 128;
#ifdef LARTPC_DEBUG_CLOCKS
__device__ unsigned long long g_ct_dbg[16];   // measurement build: thread 0's cycles per phase of a tile
#define CT_T(x) const long long x = clock64()
#define CT_ADD(i, v) ct_acc[i] += (unsigned long long)(v)
#else
#define CT_T(x)
#define CT_ADD(i, v)
#endif
#ifndef LARTPC_CT_KB
#define LARTPC_CT_KB 64
#endif
#ifndef LARTPC_CT_CTAS
#define LARTPC_CT_CTAS 4
#endif
// 64 columns per batch and four CTAs per SM.  48 and five (44 KB of shared memory and 96 registers each) were measured: hit
// lists bit-identical, charge lattice 62.2 -> 60.3 - 61.2 ms at configs[3] (under the power cap), but 5 - 10 % SLOWER at every
// point of the configs[4] sweep (n = 1e7: 58.1 -> 64.1 ms; base 0.856 -> 0.918 ms): dense tiles pay per batch
constexpr int CT_KB = LARTPC_CT_KB;                      // samples per batch (a multiple of 16, at most 64: one thread of a role per column)
static_assert(CT_KB % 16 == 0 && CT_KB >= 16 && CT_KB <= 64, "operand columns of a batch");
constexpr int CT_A_HALF = 128 * CT_KB * 2;             // bytes of one precision half of the WXY operand (16 KB)
constexpr int CT_B_HALF = 64 * CT_KB * 2;              // ... of the WT operand (8 KB)
// per-segment record of the splat, written once per S4 call (coalesced) and gathered by the tiles
struct __align__(16) SegRec {
    double ub_s, ub_e, vb_s, vb_e;      // end points on the plane in LUT bins
    double tk_s, tk_e;                  // arrival times in ticks from t_origin
    float isT, ist, qa, rho;            // 1 / (sqrt 2 sigma) in bins and ticks, Q_a, extent over sigma (node-rule choice)
    int N, a_lo, a_hi, b_lo, b_hi, jt0, jt1, flags;   // flags: segment id << 1 | (sigma = 0)
};
static_assert(sizeof(SegRec) == SEG_REC_BYTES && offsetof(SegRec, N) == SEG_REC_BOX_OFFSET && offsetof(SegRec, jt1) == SEG_REC_BOX_OFFSET + 24,
              "SegRec is six 16-byte chunks; the plan's tile classes read its last two (common.cuh)");
constexpr int CT_CTL = 1024;                           // barriers, scratch, tile ring, prefetched ids
constexpr int CT_SMEM = 2 * CT_A_HALF + 2 * CT_B_HALF + 128 + CT_CTL + sizeof(SegLocal) * SEGCAP + sizeof(SegRec) * SEGCAP;

// MN-major canonical layout: element (mn, k) of an operand with G groups of 8 along MN:
//   (mn % 8) * 2 + (k % 8) * 16 + (mn / 8) * 128 [SBO] + (k / 8) * 128 * G [LBO]   bytes
__device__ __forceinline__ uint32_t ct_col_offset(int k, int G) { return (uint32_t)((k & 7) * 16 + (k >> 3) * 128 * G); }

__device__ __forceinline__ void split_store8(unsigned char *hi, unsigned char *lo, const float (&x)[8])
{
    __half2 h[4], l[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        h[i] = __floats2half2_rn(x[2 * i], x[2 * i + 1]);
        const float2 f = __half22float2(h[i]);
        l[i] = __floats2half2_rn(x[2 * i] - f.x, x[2 * i + 1] - f.y);
    }
    *(uint4 *)hi = *(const uint4 *)h;
    *(uint4 *)lo = *(const uint4 *)l;
}

// erf(x) = sign(x) (1 - 2^(-t P(t))), t = min(|x|, 4.2): one branch-free formula, P a degree-7 fit of -log2(erfc(t)) / t
// weighted by t erfc(t) (iteratively re-weighted least squares; checked against scipy.special.erf: |error| <= 1.1e-7 ABSOLUTE over the whole line, float32
// evaluation included).  The weights are differences of erf at neighbouring edges, so absolute accuracy is what counts;
// erff() spends twice the instructions on relative accuracy near 0 that the difference throws away.
__device__ __forceinline__ float erf_fast(float x)
{
    const float t = fminf(fabsf(x), 4.2f);
    float pp = 4.535783592e-05f;
    pp = fmaf(pp, t, -4.455014132e-04f);
    pp = fmaf(pp, t, 1.489421586e-03f);
    pp = fmaf(pp, t, 7.746618357e-04f);
    pp = fmaf(pp, t, -2.825370803e-02f);
    pp = fmaf(pp, t, 1.484816223e-01f);
    pp = fmaf(pp, t, 9.184163809e-01f);
    pp = fmaf(pp, t, 1.627908587e+00f);
    float e;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e) : "f"(-pp * t));
    return copysignf(1.0f - e, x);
}


// Node rule (quadrature_tables.cuh) for a segment, or a run of a segment's midpoints, whose extent over the diffusion
// sigma is rho and that holds n_mid midpoints: index into c_quad_n / c_quad_off, -1 = keep the midpoints.  Thresholds:
// the n-node rule reproduces the midpoint sum to a few 1e-6 of the largest cell for N = 100 and ~1e-5 for N = 50 (DESIGN.md
// section 6 has the measured table); the rules below 8 nodes are used from 32 midpoints on.
__device__ __forceinline__ int quad_rule_for(float rho, int n_mid)
{
    int k = rho <= 1.0f ? 0 : rho <= 1.75f ? 1 : rho <= 2.25f ? 2 : rho <= 3.5f ? 3 : rho <= 5.5f ? 4 : rho <= 8.f ? 5
          : rho <= 12.f ? 6 : rho <= 16.f ? 7 : -1;
    if (k >= 0 && k < 3 && n_mid < 32) k = 3;
    return (k >= 0 && n_mid >= 3 * c_quad_n[k]) ? k : -1;
}

// one thread per segment: the record the tiles gather (every division of the old per-tile staging happens here, once)
__global__ void __launch_bounds__(256)
seg_record_kernel(DevParams p, int64_t n, const float *__restrict__ q_anode, const float *__restrict__ sigma_T,
                  const float *__restrict__ sigma_t, const double *__restrict__ u_s, const double *__restrict__ v_s,
                  const double *__restrict__ u_e, const double *__restrict__ v_e, const double *__restrict__ T_s,
                  const double *__restrict__ T_e, const int32_t *__restrict__ a_lo, const int32_t *__restrict__ a_hi,
                  const int32_t *__restrict__ b_lo, const int32_t *__restrict__ b_hi, const int32_t *__restrict__ jt0,
                  const int32_t *__restrict__ jt1, const int32_t *__restrict__ n_samples, SegRec *__restrict__ rec,
                  long long *composite_flag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double inv_bin = 1.0 / p.bin, inv_dt = 1.0 / p.dt;
    SegRec r;
    r.ub_s = u_s[i] * inv_bin;  r.ub_e = u_e[i] * inv_bin;
    r.vb_s = v_s[i] * inv_bin;  r.vb_e = v_e[i] * inv_bin;
    r.tk_s = (T_s[i] - p.t_origin) * inv_dt;  r.tk_e = (T_e[i] - p.t_origin) * inv_dt;
    const float sT = sigma_T[i], st = sigma_t[i];
    const bool zero_sigma = !(sT > 0.0f) || !(st > 0.0f);
    r.isT = zero_sigma ? 0.f : (float)(p.bin * 0.70710678118654752440 / (double)sT);
    r.ist = zero_sigma ? 0.f : (float)(p.dt * 0.70710678118654752440 / (double)st);
    r.qa = q_anode[i];
    r.rho = 1.41421356f * fmaxf(fmaxf(fabsf((float)(r.ub_e - r.ub_s)), fabsf((float)(r.vb_e - r.vb_s))) * r.isT,
                                fabsf((float)(r.tk_e - r.tk_s)) * r.ist);
    r.N = n_samples[i];
    r.a_lo = a_lo[i]; r.a_hi = a_hi[i]; r.b_lo = b_lo[i]; r.b_hi = b_hi[i]; r.jt0 = jt0[i]; r.jt1 = jt1[i];
    // a segment beyond the largest rule that is long enough to be cut into runs with a rule each: the splat then runs
    // its composite instance (COMP below)
    if (!zero_sigma && r.rho > 16.f && r.N < (1 << 24) && q_anode[i] > 0.f) {
        const int pieces = min((int)ceilf(r.rho * (1.0f / 16.f)), 64);
        const float rho = r.rho / (float)pieces;
        if (quad_rule_for(rho, r.N / pieces) >= 0) *composite_flag = 1;          // (the choice stage_segment<true> makes)
    }
    r.flags = (int)(i << 1) | (zero_sigma ? 1 : 0);                  // segment id (n < 2^30) and the sigma = 0 flag
    uint4 *dst = (uint4 *)(rec + i);
    const uint4 *src = (const uint4 *)&r;
#pragma unroll
    for (int c = 0; c < 6; ++c) dst[c] = src[c];
}

// record -> tile-relative staging entry; returns the number of operand columns the segment takes in this tile
template <bool COMP>
__device__ __forceinline__ int stage_segment(const DevParams &p, const SegRec &r, int s, int NB, int A_t, int B_t, int J_t,
                                             SegLocal &L)
{
    L.seg = s;
    L.N = r.N;
    L.alo = max(r.a_lo - A_t, 0);  L.ahi = min(r.a_hi - A_t, NB - 1);
    L.blo = max(r.b_lo - B_t, 0);  L.bhi = min(r.b_hi - B_t, NB - 1);
    L.jlo = max(max(r.jt0, 0) - J_t, 0);
    L.jhi = min(min(r.jt1, p.j_max) - J_t, p.Jc - 1);
    L.as = (float)(r.ub_s - (double)A_t);  L.ae = (float)(r.ub_e - (double)A_t);
    L.bs = (float)(r.vb_s - (double)B_t);  L.be = (float)(r.vb_e - (double)B_t);
    L.ts = (float)(r.tk_s - (double)J_t);  L.te = (float)(r.tk_e - (double)J_t);
    L.zero_sigma = r.flags & 1;
    L.isT = r.isT;  L.ist = r.ist;
    L.q = r.qa / (float)r.N;                                          // eq. (3.8): Q_a / N per sample point
    // Node rule instead of the N midpoints (quadrature_tables.cuh): rho = the segment's extent over the diffusion
    // sigma, per axis, decides how many nodes reproduce the midpoint sum to ~1e-6 of the largest cell (DESIGN.md
    // section 6 has the measured errors); short or sharp segments keep their own N points.
    L.qa = r.qa;
    L.inv_n2 = 1.0f / ((float)r.N * (float)r.N);
    L.inv_n4 = L.inv_n2 * L.inv_n2;
    L.rule = -1;
    int nq = r.N;
    if (p.rnd_m > 0) nq = r.N * p.rnd_m;                              // eq. (3.9) as printed: one column per perturbed point
    else if (!L.zero_sigma) {
        // COMP: long or sharp segments are cut into `pieces` runs of consecutive midpoints (sizes differing by at most
        // one), each run with its own rule -- the identity holds run by run; L.rule then also carries the nodes per
        // piece (<< 8) and pieces - 1 (<< 16)
        const int pieces = (!COMP || r.rho <= 16.f || r.N >= (1 << 24)) ? 1 : min((int)ceilf(r.rho * (1.0f / 16.f)), 64);
        const float rho = r.rho / (float)pieces;
        const int k = quad_rule_for(rho, r.N / pieces);
        if (k >= 0) {
            L.rule = c_quad_off[k];
            nq = pieces * c_quad_n[k];
            if (COMP) L.rule |= (c_quad_n[k] << 8) | ((pieces - 1) << 16);
        }
    }
    return (L.jlo > L.jhi || L.alo > L.ahi || L.blo > L.bhi) ? 0 : nq;  // box misses this tile: no columns
}

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"(rtc::s32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async8(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(rtc::s32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async4(void *smem, const void *gmem)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(rtc::s32(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }

template <int NB, bool RND, bool COMP>   // RND: eq. (3.9) as printed, p.rnd_m random perturbations per sample point
                                        // COMP: composite node rules for segments beyond the largest rule
__global__ void __launch_bounds__(CT_THREADS, LARTPC_CT_CTAS) charge_lattice_tc_kernel(const SplatArgs a)
{
    extern __shared__ unsigned char smem_dyn[];
    const DevParams &p = a.p;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int NB2 = NB * NB;
    constexpr int MG = 16, NG = 8;                                   // groups of 8 along M (128 cells) and N (64 ticks)
    const uint32_t sbase = (rtc::s32(smem_dyn) + 127u) & ~127u;
    unsigned char *base = smem_dyn + (sbase - rtc::s32(smem_dyn));
    unsigned char *Ahi = base, *Alo = base + CT_A_HALF, *Bhi = base + 2 * CT_A_HALF, *Blo = Bhi + CT_B_HALF;
    unsigned char *ctl = Blo + CT_B_HALF;                            // mbarrier, TMEM pointer, reduction scratch
    const uint32_t bar = sbase + 2 * CT_A_HALF + 2 * CT_B_HALF, tptr_addr = bar + 8;
    volatile uint32_t *tptr = (volatile uint32_t *)(ctl + 8);
    float *red = (float *)(ctl + 16);                                // [4] max, then ints
    int *redi = (int *)(ctl + 32);                                   // [4][4] lo, hi, non-zero cells of blocks 0 1 | 2 3
    int *pre = (int *)(ctl + 96);                                    // [SEGCAP + 1] running column counts
    volatile int *s_q = (volatile int *)(ctl + 240);                 // ring of 3: this tile, the next, the one after
    TileDesc *s_td = (TileDesc *)(ctl + 256);                        // [3] their descriptors
    int2 *s_tl = (int2 *)(ctl + 304);                                // [3] their segment lists {start, count}
    int *s_pid = (int *)(ctl + 336);                                 // [SEGCAP] segment ids of the next tile's first chunk
    unsigned long long *s_cnt = (unsigned long long *)(ctl + 480);   // [3] this CTA's work counters, added to the global ones once
    SegLocal *segs = (SegLocal *)(ctl + CT_CTL);
    SegRec *s_rec = (SegRec *)(ctl + CT_CTL + sizeof(SegLocal) * SEGCAP);   // records of the next tile's first chunk
    const SegRec *rec = (const SegRec *)a.rec;

    if (tid == 0) {
        s_cnt[0] = s_cnt[1] = s_cnt[2] = 0ull;
        rtc::mbar_init(bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const int q0 = atomicAdd(a.work, 1), q1 = atomicAdd(a.work, 1), q2 = atomicAdd(a.work, 1);
        s_q[0] = q0;  s_q[1] = q1;  s_q[2] = q2;
        if (q0 < a.n_tiles) { s_td[0] = a.tile_desc[q0];  s_tl[0] = a.tile_list[q0]; }
        if (q1 < a.n_tiles) { s_td[1] = a.tile_desc[q1];  s_tl[1] = a.tile_list[q1]; }
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tptr_addr), "r"(64u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    // cell rows NB2 .. 127 of the WXY operand are never written: zero the whole operand once per CTA
    for (int i = tid; i < 2 * CT_A_HALF / 16; i += CT_THREADS) ((uint4 *)Ahi)[i] = make_uint4(0u, 0u, 0u, 0u);
    rtc::tc_fence_before();
    __syncthreads();
    rtc::tc_fence_after();
    const uint32_t tmem = *tptr;
    // instruction descriptor: D fp32, A / B fp16, both MN-major, N = 64, M = 128
    const uint32_t idesc = (1u << 4) | (1u << 15) | (1u << 16) | ((uint32_t)(64 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);

    const int s_in = tid & 63;                                       // sample column of this thread
    const bool role_a = tid < 64;                                    // warps 0-1: WXY, warps 2-3: WT
    uint32_t mma_phase = 0;
    int slot = 0;                                                    // ring position of the current tile
    bool have_rec = false;                                           // s_rec holds the first chunk of the current tile

#ifdef LARTPC_DEBUG_CLOCKS
    unsigned long long ct_acc[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
#endif
    while (true) {
#ifdef LARTPC_DEBUG_CLOCKS
        long long c_top = clock64();
#endif
        const int tile = s_q[slot];
        if (tile >= a.n_tiles) break;                                // CTA-uniform: the ring is read after a barrier
        const TileDesc td = s_td[slot];
        const int2 tl = s_tl[slot];
        const int s1 = slot == 2 ? 0 : slot + 1, s2 = s1 == 2 ? 0 : s1 + 1;
        const int tile1 = s_q[s1], tile2 = s_q[s2];
        const int A_t = td.px * NB, B_t = td.py * NB, J_t = td.j_start;
        const int lstart = tl.x, lcount = tl.y;
        const int bm = __ldg(a.tb_mask + tile / TC_UNIT_TILES);          // for the read-out, in flight until then
        int q_new = 0;
        bool any_mma = false, fetched = false;

        // records of the next tile: issued once the ids asked for at the top of this tile have had time to land
        auto fetch_next_records = [&]() {
            cp_async_wait_all();
            __syncwarp();
            if (tile1 < a.n_tiles && lane < min(SEGCAP, s_tl[s1].y)) {
                const uint4 *src = (const uint4 *)(rec + s_pid[lane]);
                uint4 *dst = (uint4 *)(s_rec + lane);
#pragma unroll
                for (int c = 0; c < 6; ++c) cp_async16(dst + c, src + c);
            }
        };

        for (int l0 = 0; l0 < lcount; l0 += SEGCAP) {
            if (l0 > 0) __syncthreads();
            const int nseg = min(SEGCAP, lcount - l0);
            // The K dimension of the contraction is "sample", whichever segment it belongs to: the columns of the staged
            // segments are laid end to end (pre[] = running sum of their counts, in list order) and cut into batches of 64.
            CT_T(c_s0);
            if (warp == 0) {
                int n_eff = 0;
                if (lane < nseg) {
                    SegRec r;
                    if (l0 == 0 && have_rec) r = s_rec[lane];
                    else {
                        const uint4 *src = (const uint4 *)(rec + a.pair_seg[lstart + l0 + lane]);
                        uint4 *dst = (uint4 *)&r;
#pragma unroll
                        for (int c = 0; c < 6; ++c) dst[c] = __ldg(src + c);
                    }
                    SegLocal L;
                    n_eff = stage_segment<COMP>(p, r, r.flags >> 1, NB, A_t, B_t, J_t, L);
                    segs[lane] = L;
                }
                int inc = n_eff;
                for (int d = 1; d < 32; d <<= 1) {
                    const int o = __shfl_up_sync(0xffffffffu, inc, d);
                    if (lane >= d) inc += o;
                }
                pre[lane + 1] = inc;
                if (lane == 0) pre[0] = 0;
            }
            CT_T(c_s1);
            __syncthreads();
            CT_T(c_staged);  CT_ADD(0, c_staged - c_top);  CT_ADD(8, c_s0 - c_top);  CT_ADD(9, c_s1 - c_s0);  CT_ADD(10, c_staged - c_s1);  CT_ADD(11, 1);
            if (l0 == 0 && warp == 0) {
                // look-ahead: cursor for the tile three ahead, descriptor of the tile two ahead, ids of the next tile
                if (lane == 0) {
                    q_new = atomicAdd(a.work, 1);
                    if (tile2 < a.n_tiles) { cp_async16(&s_td[s2], a.tile_desc + tile2);  cp_async8(&s_tl[s2], a.tile_list + tile2); }
                }
                if (tile1 < a.n_tiles) {
                    const int2 t1 = s_tl[s1];
                    if (lane < min(SEGCAP, t1.y)) cp_async4(&s_pid[lane], a.pair_seg + t1.x + lane);
                }
            }
            const int total = pre[nseg];
            if (tid == 0 && total) {
                s_cnt[1] += (unsigned long long)total;                               // (thread 0 alone writes these two)
                s_cnt[2] += 3ull * (unsigned long long)((total + 15) / 16);         // hi hi + hi lo + lo hi per 16 columns
            }
            for (int s0 = 0; s0 < total; s0 += CT_KB) {
                CT_T(c_b0);
                const int nsb = min(CT_KB, total - s0), nk16 = (nsb + 15) >> 4;
                if (s_in < 16 * nk16) {
                    const bool real = s_in < nsb;
                    const int slot = s0 + min(s_in, nsb - 1);
                    int li = 0;                                           // last li with pre[li] <= slot (SEGCAP = 32)
    #pragma unroll
                    for (int step = 16; step; step >>= 1)
                        if (li + step < nseg && pre[li + step] <= slot) li += step;
                    const SegLocal L = segs[li];
                    int mu = slot - pre[li], nu = 0;
                    if (RND) { nu = mu % p.rnd_m;  mu /= p.rnd_m; }                 // column = perturbation nu of sample point mu
                    float f = ((float)mu + 0.5f) * (1.0f / (float)L.N), qw = L.q;   // position along the segment, charge
                    if (RND) qw = L.q / (float)p.rnd_m;                            // Q_a / (N M)
                    else if (L.rule >= 0) {
                        if (!COMP || (L.rule >> 16) == 0) {
                            const float4 r = __ldg(&g_quad[(COMP ? (L.rule & 0xff) : L.rule) + mu]);
                            f = r.x;
                            qw = L.qa * (r.y - r.z * L.inv_n2 + r.w * L.inv_n4);
                        } else {
                            // column mu = node i of piece pc; the piece holds midpoints [s_p, e_p) of the segment's N
                            // (N < 2^24 there: 32-bit products)
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
                    // sigma = 0: the bin / tick is an integer decision taken in float64 in the oracle's order
                    int ia = -1, ib = -1, jj = -1;
                    if ((RND || L.zero_sigma) && real) {
                        const int s = L.seg;
                        const double fd = xdiv(xadd((double)mu, 0.5), (double)L.N);
                        double z[3] = {0.0, 0.0, 0.0}, sT = 0.0, st = 0.0;
                        if (RND) {
                            perturbation_normals(p.rnd_seed, (uint32_t)s, (uint32_t)mu, (uint32_t)nu, p.n_sigma_map, z);
                            sT = (double)a.sigma_T[s];  st = (double)a.sigma_t[s];
                        }
                        if (role_a) {
                            const double us = a.u_s[s], ue = a.u_e[s], vs = a.v_s[s], ve = a.v_e[s];
                            const double uu = xadd(xadd(us, xmul(xsub(ue, us), fd)), xmul(sT, z[0]));
                            const double vv = xadd(xadd(vs, xmul(xsub(ve, vs), fd)), xmul(sT, z[1]));
                            const long long xa = (long long)floor(xdiv(uu, p.bin)) - A_t;
                            const long long xb = (long long)floor(xdiv(vv, p.bin)) - B_t;
                            if (xa >= 0 && xa < NB && xb >= 0 && xb < NB) { ia = (int)xa; ib = (int)xb; }
                        } else {
                            const double Ts = a.T_s[s], Te = a.T_e[s];
                            const double TT = xadd(xadd(Ts, xmul(xsub(Te, Ts), fd)), xmul(st, z[2]));
                            long long j = (long long)floor(xdiv(xsub(TT, p.t_origin), p.dt));
                            if (j >= 0 && j <= p.j_max && j - J_t >= 0 && j - J_t < p.Jc) jj = (int)(j - J_t);
                        }
                    }
                    if (role_a) {
                        float wx[NB], wy[NB];
                        if (!real) {
    #pragma unroll
                            for (int i = 0; i < NB; ++i) wx[i] = wy[i] = 0.f;
                        } else if (RND || L.zero_sigma) {
    #pragma unroll
                            for (int i = 0; i < NB; ++i) { wx[i] = (i == ia) ? 1.f : 0.f; wy[i] = (i == ib) ? 1.f : 0.f; }
                        } else {
                            const float px = fmaf(L.ae - L.as, f, L.as), py = fmaf(L.be - L.bs, f, L.bs);
                            float ex = erf_fast((0.f - px) * L.isT), ey = erf_fast((0.f - py) * L.isT);
    #pragma unroll
                            for (int i = 0; i < NB; ++i) {
                                const float ex1 = erf_fast(((float)(i + 1) - px) * L.isT), ey1 = erf_fast(((float)(i + 1) - py) * L.isT);
                                wx[i] = (i >= L.alo && i <= L.ahi) ? 0.5f * (ex1 - ex) : 0.f;
                                wy[i] = (i >= L.blo && i <= L.bhi) ? 0.5f * (ey1 - ey) : 0.f;
                                ex = ex1;  ey = ey1;
                            }
                        }
                        const uint32_t col = ct_col_offset(s_in, MG);
    #pragma unroll
                        for (int g = 0; g < (NB2 + 7) / 8; ++g) {
                            float x[8];
    #pragma unroll
                            for (int i = 0; i < 8; ++i) {
                                const int m = 8 * g + i;
                                x[i] = m < NB2 ? wx[m % NB] * wy[m / NB] : 0.f;
                            }
                            split_store8(Ahi + col + 128 * g, Alo + col + 128 * g, x);
                        }
                    } else {
                        const uint32_t col = ct_col_offset(s_in, NG);
                        const float pt = fmaf(L.te - L.ts, f, L.ts);
                        const float hq = 0.5f * qw;
                        for (int g = 0; g < NG; ++g) {
                            float x[8];
                            const int j0 = 8 * g;
                            if (!real || j0 + 7 < L.jlo || j0 > L.jhi) {
    #pragma unroll
                                for (int i = 0; i < 8; ++i) x[i] = 0.f;
                            } else if (RND || L.zero_sigma) {
    #pragma unroll
                                for (int i = 0; i < 8; ++i) x[i] = (j0 + i == jj) ? qw : 0.f;
                            } else {
                                float e0 = erf_fast(((float)j0 - pt) * L.ist);
    #pragma unroll
                                for (int i = 0; i < 8; ++i) {
                                    const float e1 = erf_fast(((float)(j0 + i + 1) - pt) * L.ist);
                                    x[i] = (j0 + i >= L.jlo && j0 + i <= L.jhi) ? hq * (e1 - e0) : 0.f;
                                    e0 = e1;
                                }
                            }
                            split_store8(Bhi + col + 128 * g, Blo + col + 128 * g, x);
                        }
                    }
                }
                // operands written by the generic proxy, read by the tensor core (async proxy)
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                CT_T(c_b1);
                __syncthreads();
                CT_T(c_b2);
                if (tid == 0) {
                    rtc::tc_fence_after();
                    for (int k16 = 0; k16 < nk16; ++k16) {
                        const uint32_t ao = 2 * k16 * 128 * MG, bo = 2 * k16 * 128 * NG;
                        const uint64_t ah = rtc::smem_desc(sbase + ao, 128 * MG, 128, 0);
                        const uint64_t al = rtc::smem_desc(sbase + CT_A_HALF + ao, 128 * MG, 128, 0);
                        const uint64_t bh = rtc::smem_desc(sbase + 2 * CT_A_HALF + bo, 128 * NG, 128, 0);
                        const uint64_t bl = rtc::smem_desc(sbase + 2 * CT_A_HALF + CT_B_HALF + bo, 128 * NG, 128, 0);
                        rtc::tc_mma_f16(tmem, ah, bh, idesc, (any_mma || k16) ? 1u : 0u);
                        rtc::tc_mma_f16(tmem, ah, bl, idesc, 1u);
                        rtc::tc_mma_f16(tmem, al, bh, idesc, 1u);
                    }
                    rtc::tc_commit(bar);
                }
                if (!fetched && warp == 0) fetch_next_records();
                fetched = true;
                any_mma = true;
                rtc::mbar_wait(bar, mma_phase);                        // the MMAs have read the operands (and landed)
                mma_phase ^= 1u;
                CT_T(c_b3);  CT_ADD(1, c_b1 - c_b0);  CT_ADD(2, c_b2 - c_b1);  CT_ADD(3, c_b3 - c_b2);  CT_ADD(6, 1);
#ifdef LARTPC_DEBUG_CLOCKS
                c_top = c_b3;                                          // (a further chunk's staging counts from here)
#endif
            }
        }
        if (!fetched && warp == 0) fetch_next_records();
        CT_T(c_r0);
        // ------------------------------------------------------------------ accumulator -> operand image of the response
        if (!any_mma) {                                                   // CTA-uniform: no segment reaches this window
            if (tid == 0) *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(1, 0, 0, 0);
        } else {
            rtc::tc_fence_after();
            uint32_t v[2][32];
            const uint32_t tlane = tmem + ((uint32_t)(32 * warp) << 16);  // thread = cell row m = tid
            rtc::tmem_ld32(tlane, v[0]);
            rtc::tmem_ld32(tlane + 32, v[1]);
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            float mx = 0.f;
            uint32_t nz_lo = 0u, nz_hi = 0u;                             // bit j: tick j of this row holds charge
    #pragma unroll
            for (int j = 0; j < 64; ++j) {
                const float x = __uint_as_float(v[j >> 5][j & 31]);
                mx = fmaxf(mx, fabsf(x));
                if (x != 0.f) { if (j < 32) nz_lo |= 1u << j; else nz_hi |= 1u << (j - 32); }
            }
            int lo = nz_lo ? __ffs(nz_lo) - 1 : nz_hi ? 31 + __ffs(nz_hi) : INT_MAX;
            int hi = nz_hi ? 63 - __clz(nz_hi) : nz_lo ? 31 - __clz(nz_lo) : -1;
            // non-zero cells of this row per 16-tick block, 16 bits each
            int pk01 = __popc(nz_lo & 0xffffu) | __popc(nz_lo >> 16) << 16, pk23 = __popc(nz_hi & 0xffffu) | __popc(nz_hi >> 16) << 16;
            for (int d = 16; d; d >>= 1) {
                mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, d));
                lo = min(lo, __shfl_xor_sync(0xffffffffu, lo, d));
                hi = max(hi, __shfl_xor_sync(0xffffffffu, hi, d));
                pk01 += __shfl_xor_sync(0xffffffffu, pk01, d);           // <= 32 x 16 per field and warp, <= 1600 per tile
                pk23 += __shfl_xor_sync(0xffffffffu, pk23, d);
            }
            if (lane == 0) { red[warp] = mx; redi[4 * warp] = lo; redi[4 * warp + 1] = hi; redi[4 * warp + 2] = pk01; redi[4 * warp + 3] = pk23; }
            __syncthreads();
    #pragma unroll
            for (int w = 0; w < CT_THREADS / 32; ++w) {
                mx = w ? fmaxf(mx, red[w]) : red[0];
                lo = w ? min(lo, redi[4 * w]) : redi[0];
                hi = w ? max(hi, redi[4 * w + 1]) : redi[1];
                pk01 = w ? pk01 + redi[4 * w + 2] : redi[2];
                pk23 = w ? pk23 + redi[4 * w + 3] : redi[3];
            }
            const int nzb0 = pk01 & 0xffff, nzb1 = pk01 >> 16, nzb2 = pk23 & 0xffff, nzb3 = pk23 >> 16;
            const int nz = nzb0 + nzb1 + nzb2 + nzb3;
            // what the response's epilogue needs to add back the expected truncation loss of the tensor-core accumulation
            // (response_tc.cuh "Accuracy"): non-zero cells per 16-tick block, in units of 8 cells, one byte per block
            const int nz_packed = min((nzb0 + 4) >> 3, 255) | min((nzb1 + 4) >> 3, 255) << 8 | min((nzb2 + 4) >> 3, 255) << 16 |
                                  min((nzb3 + 4) >> 3, 255) << 24;
            int e = 0;
            if (mx >= 32768.f) e = min(((__float_as_int(mx) >> 23) & 0xff) - 127 - 14, 100);   // mx * 2^-e in [2^14, 2^15)
            if (!(mx < 3.0e38f)) e = 0;                                   // inf / nan charge: leave it visible
            const float sc = __int_as_float((127 - e) << 23);
            if (tid == CT_THREADS - 1) {                                  // a lane whose cell row does not exist: off the stores' path
                if (nz == 0) *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(1, 0, 0, 0);
                else {
                    *(int4 *)(a.tile_range + TILE_META * tile) = make_int4(lo / RESP_NO, (hi + p.K - 1) / RESP_NO, e, nz_packed);
                    // multiply-adds the method needs here: non-zero cells x in-plane targets x K
                    const DevTpc &tp = a.tpcs[td.tpc];
                    const int vx = min(td.px + p.H, tp.nx - 1) - max(td.px - p.H, 0) + 1;
                    const int vy = min(td.py + p.H, tp.ny - 1) - max(td.py - p.H, 0) + 1;
                    if (vx > 0 && vy > 0) s_cnt[0] += (unsigned long long)nz * (unsigned long long)(vx * vy * p.K);   // (this thread alone)
                }
            }
            {
                // blocks this cell row charges -> the unit's per-bin block mask the response skips by (4 bits per bin, 8 bins
                // per word: the 8 lanes of a word combine first, one atomic per word and tile)
                int bits = ((nz_lo & 0xffffu) ? 1 : 0) | ((nz_lo >> 16) ? 2 : 0) | ((nz_hi & 0xffffu) ? 4 : 0) | ((nz_hi >> 16) ? 8 : 0);
                bits <<= 4 * (lane & 7);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 1);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 2);
                bits |= __shfl_xor_sync(0xffffffffu, bits, 4);
                if ((lane & 7) == 0 && bits) atomicOr(a.cmask + (size_t)(tile / TC_UNIT_TILES) * TC_CMASK_WORDS + (tid >> 3), bits);
            }
            if (tid < NB2) {
                // rows of the response's operand image; only the 16-tick blocks some tile of the block charges exist
                const int tb = tile / rtc::TB, r = tile - tb * rtc::TB;
                unsigned char *cb = (unsigned char *)a.charge + ((size_t)tb * NB2 + tid) * (rtc::NBLK * rtc::A_BLOCK_BYTES);
#pragma unroll
                for (int b = 0; b < rtc::NBLK; ++b) {
                    if (!(bm >> b & 1)) continue;
                    float x[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) x[i] = __uint_as_float(v[(16 * b + i) >> 5][(16 * b + i) & 31]) * sc;
                    rtc::store_a_block16(cb + b * rtc::A_BLOCK_BYTES, r, x);
                }
            }
        }
        CT_T(c_r1);
        // the look-ahead of this tile has landed; hand the ring on
        if (warp == 0) {
            cp_async_wait_all();
            if (lane == 0) s_q[slot] = q_new;
        }
        have_rec = tile1 < a.n_tiles;
        slot = s1;
        rtc::tc_fence_before();
        __syncthreads();
        rtc::tc_fence_after();
        CT_T(c_end);  CT_ADD(4, c_r1 - c_r0);  CT_ADD(5, c_end - c_r1);  CT_ADD(7, 1);
    }
#ifdef LARTPC_DEBUG_CLOCKS
    if (tid == 0) for (int i = 0; i < 16; ++i) atomicAdd(&g_ct_dbg[i], ct_acc[i]);
#endif
    rtc::tc_fence_before();
    __syncthreads();
    if (tid == 0) {                                                  // one atomic per counter and CTA, not per tile
        if (s_cnt[0]) atomicAdd(a.fma_counter, s_cnt[0]);
        if (s_cnt[1]) atomicAdd(a.fma_counter + 3, s_cnt[1]);
        if (s_cnt[2]) atomicAdd(a.fma_counter + 4, s_cnt[2]);
    }
    if (warp == 0) {
        rtc::tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(64u) : "memory");
    }
}
