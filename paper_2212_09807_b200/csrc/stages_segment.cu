// S1 quench, S2 drift, S3 pixel mapping + tile plan: one thread per segment,
// structure-of-arrays float32 inputs read with coalesced 128-bit loads where alignment allows.
// These stages are HBM-bound; arithmetic per segment is a few dozen operations.
#include "common.cuh"
#include "scan.cuh"

// -------------------------------------------------------------------------------------------------
// S1  recombination, eqs. (3.1)/(3.2) P:L575-583.  float32 arithmetic.
// -------------------------------------------------------------------------------------------------
__device__ __forceinline__ void quench_one(const DevParams &p, float dx, float dy, float dz, float dE,
                                           float &dEdx, float &n_e)
{
    float L = sqrtf(fmaf(dz, dz, fmaf(dy, dy, dx * dx)));
    if (!(L > 0.0f) || !(dE > 0.0f)) { dEdx = 0.0f; n_e = 0.0f; return; }
    float q = dE / L;
    float R;
    if (p.recomb_model == 0) {
        R = (float)p.birks_ab / (1.0f + (float)(p.birks_kb / p.eps) * q);           // eq. (3.1)
    } else {
        float xi = (float)(p.box_beta / p.eps) * q;
        R = fmaxf(logf((float)p.box_alpha + xi) / xi, 0.0f);                          // eq. (3.2), D6
    }
    dEdx = q;
    n_e = R * (dE * (float)(1.0 / p.w_ion));
}

template <int VEC>
__global__ void __launch_bounds__(256) quench_kernel(DevParams p, SegPtrs s, int64_t n, float *dEdx, float *n_e)
{
    int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    if (i >= n) return;
    if (VEC == 4 && i + 3 < n) {
        float4 xs = *(const float4 *)(s.xs + i), ys = *(const float4 *)(s.ys + i), zs = *(const float4 *)(s.zs + i);
        float4 xe = *(const float4 *)(s.xe + i), ye = *(const float4 *)(s.ye + i), ze = *(const float4 *)(s.ze + i);
        float4 de = *(const float4 *)(s.dE + i);
        float4 o1, o2;
        quench_one(p, xe.x - xs.x, ye.x - ys.x, ze.x - zs.x, de.x, o1.x, o2.x);
        quench_one(p, xe.y - xs.y, ye.y - ys.y, ze.y - zs.y, de.y, o1.y, o2.y);
        quench_one(p, xe.z - xs.z, ye.z - ys.z, ze.z - zs.z, de.z, o1.z, o2.z);
        quench_one(p, xe.w - xs.w, ye.w - ys.w, ze.w - zs.w, de.w, o1.w, o2.w);
        *(float4 *)(dEdx + i) = o1;
        *(float4 *)(n_e + i) = o2;
    } else {
        for (int k = 0; k < VEC && i + k < n; ++k) {
            int64_t j = i + k;
            quench_one(p, s.xe[j] - s.xs[j], s.ye[j] - s.ys[j], s.ze[j] - s.zs[j], s.dE[j], dEdx[j], n_e[j]);
        }
    }
}

static bool aligned16(const void *p) { return ((uintptr_t)p & 15u) == 0; }

int launch_quench(lartpc_sim *sim, const lartpc_segments_t *seg, int64_t n, float *dEdx, float *n_e, cudaStream_t st)
{
    if (n == 0) return LARTPC_OK;
    SegPtrs s{seg->xs, seg->ys, seg->zs, seg->ts, seg->xe, seg->ye, seg->ze, seg->te, seg->dE};
    bool vec = aligned16(s.xs) && aligned16(s.ys) && aligned16(s.zs) && aligned16(s.xe) && aligned16(s.ye) &&
               aligned16(s.ze) && aligned16(s.dE) && aligned16(dEdx) && aligned16(n_e);
    if (vec) {
        ++g_lartpc_launches;
        quench_kernel<4><<<div_up(div_up(n, 4), 256), 256, 0, st>>>(sim->dp, s, n, dEdx, n_e);
    } else {
        ++g_lartpc_launches;
        quench_kernel<1><<<div_up(n, 256), 256, 0, st>>>(sim->dp, s, n, dEdx, n_e);
    }
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// -------------------------------------------------------------------------------------------------
// S2  transport, eqs. (3.3)-(3.5) P:L599-616.  The index path (TPC, distances, times, sigma) is float64
// with individually rounded operations in the order DESIGN.md fixes, because S3 turns them into integers.
// -------------------------------------------------------------------------------------------------
struct DriftCore {
    int tpc;
    double t_mid, sigma_T, sigma_t, u_s, v_s, u_e, v_e, T_s, T_e;
};

__device__ __forceinline__ int find_tpc(const DevParams &p, const DevTpc *__restrict__ tpcs, double xm, double ym,
                                        double zm)
{
    for (int k = 0; k < p.n_tpcs; ++k) {
        const DevTpc &t = tpcs[k];
        double dm = xmul((double)t.sign, xsub(zm, t.z_anode));
        if (xm >= t.x0 && xm < t.x1 && ym >= t.y0 && ym < t.y1 && dm >= 0.0 && dm <= t.drift_len) return k;
    }
    return -1;
}

__device__ __forceinline__ void drift_core(const DevParams &p, const DevTpc *__restrict__ tpcs, int tpc,
                                           float xs, float ys, float zs, float ts, float xe, float ye, float ze,
                                           float te, DriftCore &o)
{
    const DevTpc &t = tpcs[tpc];
    double zm = xmul(0.5, xadd((double)zs, (double)ze));
    o.tpc = tpc;
    o.t_mid = xdiv(drift_dist(t, zm), p.v_drift);
    o.sigma_T = xsqrt(xmul(xmul(2.0, p.d_tran), o.t_mid));
    double sigma_L = xsqrt(xmul(xmul(2.0, p.d_long), o.t_mid));
    o.sigma_t = xdiv(sigma_L, p.v_drift);
    o.u_s = xsub((double)xs, t.x0);  o.v_s = xsub((double)ys, t.y0);
    o.u_e = xsub((double)xe, t.x0);  o.v_e = xsub((double)ye, t.y0);
    o.T_s = xadd((double)ts, xdiv(drift_dist(t, (double)zs), p.v_drift));
    o.T_e = xadd((double)te, xdiv(drift_dist(t, (double)ze), p.v_drift));
}

__global__ void __launch_bounds__(256) drift_kernel(DevParams p, const DevTpc *__restrict__ tpcs, SegPtrs s,
                                                    int64_t n, const float *__restrict__ n_e, lartpc_drifted_t o)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float xs = s.xs[i], ys = s.ys[i], zs = s.zs[i], ts = s.ts[i];
    float xe = s.xe[i], ye = s.ye[i], ze = s.ze[i], te = s.te[i];
    double xm = xmul(0.5, xadd((double)xs, (double)xe));
    double ym = xmul(0.5, xadd((double)ys, (double)ye));
    double zm = xmul(0.5, xadd((double)zs, (double)ze));
    int tpc = find_tpc(p, tpcs, xm, ym, zm);
    o.tpc[i] = tpc;
    if (tpc < 0) {
        o.q_anode[i] = 0.0f; o.sigma_T[i] = 0.0f; o.sigma_t[i] = 0.0f;
        o.u_s[i] = o.v_s[i] = o.u_e[i] = o.v_e[i] = o.T_s[i] = o.T_e[i] = 0.0;
        return;
    }
    DriftCore c;
    drift_core(p, tpcs, tpc, xs, ys, zs, ts, xe, ye, ze, te, c);
    o.q_anode[i] = (float)((double)n_e[i] * exp(-c.t_mid / p.lifetime));              // eq. (3.4)
    o.sigma_T[i] = (float)c.sigma_T;                                                   // eq. (3.5)
    o.sigma_t[i] = (float)c.sigma_t;
    o.u_s[i] = c.u_s; o.v_s[i] = c.v_s; o.u_e[i] = c.u_e; o.v_e[i] = c.v_e;
    o.T_s[i] = c.T_s; o.T_e[i] = c.T_e;
}

int launch_drift(lartpc_sim *sim, const lartpc_segments_t *seg, int64_t n, const float *n_e, lartpc_drifted_t *out,
                 cudaStream_t st)
{
    if (n == 0) return LARTPC_OK;
    SegPtrs s{seg->xs, seg->ys, seg->zs, seg->ts, seg->xe, seg->ye, seg->ze, seg->te, seg->dE};
    ++g_lartpc_launches;
    drift_kernel<<<div_up(n, 256), 256, 0, st>>>(sim->dp, sim->d_tpcs, s, n, n_e, *out);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// -------------------------------------------------------------------------------------------------
// S3  pixel mapping (reading D10) and the tile plan S4 runs on.
// -------------------------------------------------------------------------------------------------
struct SegBox {
    int a_lo, a_hi, b_lo, b_hi, ix0, ix1, iy0, iy1, jt0, jt1, npix, n_samples;
    int cpx0, cpx1, cpy0, cpy1, j0, j1;          // charged pixels (clamped to the +-H margin), arrival ticks in the window
    bool deposits;
};

__device__ __forceinline__ void chunk_and_cp_range(const DevParams &p, const DevTpc &t, SegBox &b)
{
    long long x0 = floor_div_ll(b.a_lo, p.nb), x1 = floor_div_ll(b.a_hi, p.nb);
    long long y0 = floor_div_ll(b.b_lo, p.nb), y1 = floor_div_ll(b.b_hi, p.nb);
    b.cpx0 = (int)max(x0, (long long)-p.H);  b.cpx1 = (int)min(x1, (long long)(t.nx - 1 + p.H));
    b.cpy0 = (int)max(y0, (long long)-p.H);  b.cpy1 = (int)min(y1, (long long)(t.ny - 1 + p.H));
    b.j0 = max(b.jt0, 0);  b.j1 = min(b.jt1, p.j_max);     // charge outside the readout window is dropped (D23)
    b.deposits = b.npix > 0 && b.j0 <= b.j1 && b.cpx0 <= b.cpx1 && b.cpy0 <= b.cpy1;
}

__device__ __forceinline__ void seg_box(const DevParams &p, const DevTpc *__restrict__ tpcs, int tpc, float q_anode,
                                        float xs, float ys, float zs, float ts, float xe, float ye, float ze, float te,
                                        SegBox &b)
{
    double dx = xsub((double)xe, (double)xs), dy = xsub((double)ye, (double)ys), dz = xsub((double)ze, (double)zs);
    double L = xsqrt(xadd(xadd(xmul(dx, dx), xmul(dy, dy)), xmul(dz, dz)));
    long long N = (long long)ceil(xdiv(L, p.sample_step));
    b.n_samples = (int)(N < 1 ? 1 : N);
    b.deposits = false;
    if (tpc < 0 || !(q_anode > 0.0f)) {
        b.a_lo = b.b_lo = 0; b.a_hi = b.b_hi = -1; b.ix0 = b.iy0 = 0; b.ix1 = b.iy1 = -1; b.jt0 = 0; b.jt1 = -1;
        b.npix = 0;
        return;
    }
    DriftCore c;
    drift_core(p, tpcs, tpc, xs, ys, zs, ts, xe, ye, ze, te, c);
    const DevTpc &t = tpcs[tpc];
    double r = xmul(p.n_sigma_map, c.sigma_T);
    double umin = fmin(c.u_s, c.u_e), umax = fmax(c.u_s, c.u_e), vmin = fmin(c.v_s, c.v_e), vmax = fmax(c.v_s, c.v_e);
    long long al = (long long)floor(xdiv(xsub(umin, r), p.bin)), ah = (long long)floor(xdiv(xadd(umax, r), p.bin));
    long long bl = (long long)floor(xdiv(xsub(vmin, r), p.bin)), bh = (long long)floor(xdiv(xadd(vmax, r), p.bin));
    b.a_lo = (int)al; b.a_hi = (int)ah; b.b_lo = (int)bl; b.b_hi = (int)bh;
    long long x0 = floor_div_ll(al, p.nb) - p.H, x1 = floor_div_ll(ah, p.nb) + p.H;
    long long y0 = floor_div_ll(bl, p.nb) - p.H, y1 = floor_div_ll(bh, p.nb) + p.H;
    if (x0 < 0) x0 = 0;
    if (y0 < 0) y0 = 0;
    if (x1 > t.nx - 1) x1 = t.nx - 1;
    if (y1 > t.ny - 1) y1 = t.ny - 1;
    b.ix0 = (int)x0; b.ix1 = (int)x1; b.iy0 = (int)y0; b.iy1 = (int)y1;
    b.npix = (x0 <= x1 && y0 <= y1) ? (int)((x1 - x0 + 1) * (y1 - y0 + 1)) : 0;
    double rt = xmul(p.n_sigma_map, c.sigma_t);
    double tmin = fmin(c.T_s, c.T_e), tmax = fmax(c.T_s, c.T_e);
    b.jt0 = (int)floor(xdiv(xsub(xsub(tmin, rt), p.t_origin), p.dt));
    b.jt1 = (int)floor(xdiv(xsub(xadd(tmax, rt), p.t_origin), p.dt));
    chunk_and_cp_range(p, t, b);
}

__device__ __forceinline__ long long warp_max_ll(long long v)
{
    for (int d = 16; d; d >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, d));
    return v;
}
__device__ __forceinline__ long long warp_sum_ll(long long v)
{
    for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

__global__ void __launch_bounds__(256)
pixmap_kernel(DevParams p, const DevTpc *__restrict__ tpcs, SegPtrs s, int64_t n, const int32_t *__restrict__ seg_tpc,
              const float *__restrict__ q_anode, int tpc_lo, int tpc_hi, lartpc_pixmap_t o,
              int32_t *pix_count, int32_t *pix_jmin, long long *counters, int reuse)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    long long m_npix = 0, m_ticks = 0, n_act = 0, n_pairs = 0;
    if (i < n) {
        int tpc = seg_tpc[i];
        SegBox b;
        if (reuse) {
            // a later TPC batch of the same input (lartpc_run_spill): the boxes are those the first batch wrote
            b.deposits = false;
            b.npix = 0;
            if (tpc >= tpc_lo && tpc < tpc_hi) {
                b.a_lo = o.a_lo[i]; b.a_hi = o.a_hi[i]; b.b_lo = o.b_lo[i]; b.b_hi = o.b_hi[i];
                b.jt0 = o.jt0[i]; b.jt1 = o.jt1[i]; b.npix = o.npix[i];
                if (b.npix > 0) chunk_and_cp_range(p, tpcs[tpc], b);
            }
        } else {
            seg_box(p, tpcs, tpc, q_anode[i], s.xs[i], s.ys[i], s.zs[i], s.ts[i], s.xe[i], s.ye[i], s.ze[i], s.te[i], b);
            o.a_lo[i] = b.a_lo; o.a_hi[i] = b.a_hi; o.b_lo[i] = b.b_lo; o.b_hi[i] = b.b_hi;
            o.ix0[i] = b.ix0; o.ix1[i] = b.ix1; o.iy0[i] = b.iy0; o.iy1[i] = b.iy1;
            o.jt0[i] = b.jt0; o.jt1[i] = b.jt1; o.npix[i] = b.npix; o.n_samples[i] = b.n_samples;
        }
        if (b.npix > 0) {
            m_npix = b.npix;
            m_ticks = (long long)(b.jt1 - b.jt0 + 1) + p.K - 1;
            n_act = 1;
        }
        if (b.deposits && tpc >= tpc_lo && tpc < tpc_hi) {
            const DevTpc &t = tpcs[tpc];
            for (int cy = b.cpy0; cy <= b.cpy1; ++cy)
                for (int cx = b.cpx0; cx <= b.cpx1; ++cx) {
                    int cp = t.cp_base + (cy + p.H) * t.gw + (cx + p.H);
                    atomicAdd(&pix_count[cp], 1);
                    atomicMin(&pix_jmin[cp], b.j0);
                    ++n_pairs;
                }
        }
    }
    m_npix = warp_max_ll(m_npix); m_ticks = warp_max_ll(m_ticks);
    n_act = warp_sum_ll(n_act); n_pairs = warp_sum_ll(n_pairs);
    if ((threadIdx.x & 31) == 0) {
        if (m_npix) atomicMax(&counters[CNT_MAX_NPIX], m_npix);
        if (m_ticks) atomicMax(&counters[CNT_MAX_TICKS], m_ticks);
        if (n_act) atomicAdd((unsigned long long *)&counters[CNT_ACTIVE_SEGS], (unsigned long long)n_act);
        if (n_pairs) atomicAdd((unsigned long long *)&counters[CNT_PAIRS], (unsigned long long)n_pairs);
    }
}

// second pass over the segments: write the (segment, charged pixel) incidence lists
__global__ void __launch_bounds__(256)
pair_fill_kernel(DevParams p, const DevTpc *__restrict__ tpcs, int64_t n, const int32_t *__restrict__ seg_tpc,
                 lartpc_pixmap_t o, int tpc_lo, int tpc_hi, const int32_t *__restrict__ pix_start, int32_t *pix_cursor,
                 const int32_t *__restrict__ pix_jmin, unsigned long long *pix_mask,
                 int32_t *pair_seg, int64_t pair_cap, long long *counters)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int tpc = seg_tpc[i];
    if (tpc < tpc_lo || tpc >= tpc_hi) return;
    SegBox b;
    b.a_lo = o.a_lo[i]; b.a_hi = o.a_hi[i]; b.b_lo = o.b_lo[i]; b.b_hi = o.b_hi[i];
    b.jt0 = o.jt0[i]; b.jt1 = o.jt1[i]; b.npix = o.npix[i];
    if (b.npix <= 0) return;
    const DevTpc &t = tpcs[tpc];
    chunk_and_cp_range(p, t, b);
    if (!b.deposits) return;
    for (int cy = b.cpy0; cy <= b.cpy1; ++cy)
        for (int cx = b.cpx0; cx <= b.cpx1; ++cx) {
            int cp = t.cp_base + (cy + p.H) * t.gw + (cx + p.H);
            int64_t slot = (int64_t)pix_start[cp] + atomicAdd(&pix_cursor[cp], 1);
            if (slot < pair_cap) pair_seg[slot] = (int32_t)i;
            else atomicAdd((unsigned long long *)&counters[CNT_OVERFLOW], 1ull);
            // windows of Jc arrival ticks counted from the pixel's first tick (rounded down to a multiple of 4: S5 reads
            // the partial rows with aligned 16-byte loads)
            const int js = pix_jmin[cp] & ~3;
            const int w0 = min((b.j0 - js) / p.Jc, MAX_WINDOWS - 1), w1 = min((b.j1 - js) / p.Jc, MAX_WINDOWS - 1);
            for (int wd = w0 >> 6; wd <= (w1 >> 6); ++wd) {
                const int lo = max(w0 - 64 * wd, 0), hi = min(w1 - 64 * wd, 63);
                const unsigned long long m = (hi >= 63 ? ~0ull : ((1ull << (hi + 1)) - 1ull)) & ~((1ull << lo) - 1ull);
                atomicOr(&pix_mask[(size_t)cp * MASK_WORDS + wd], m);
            }
        }
}

// the atomics above fill each list in arbitrary order; sort it by segment id so that the float32
// accumulation order of S4 (and hence every output bit) is reproducible from run to run: one warp per list
constexpr int PAIR_RANK_MAX = 512;
__global__ void __launch_bounds__(128)
pair_sort_kernel(int64_t n_cells, const int32_t *__restrict__ cell_list, const int32_t *__restrict__ pix_start,
                 const int32_t *__restrict__ pix_count, int32_t *pair_seg, int64_t pair_cap)
{
    const int64_t ci = (int64_t)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    if (ci >= n_cells) return;
    const int64_t cp = cell_list[ci];
    int cnt = pix_count[cp];
    if (cnt < 2) return;
    int lane = threadIdx.x & 31;
    int64_t base = pix_start[cp];
    if (base + cnt > pair_cap) return;
    int32_t *v = pair_seg + base;
    if (cnt <= 32) {
        // one element per lane (INT32_MAX past the end), bitonic network over the warp by shuffles
        int32_t x = lane < cnt ? v[lane] : INT32_MAX;
#pragma unroll
        for (int k = 2; k <= 32; k <<= 1)
#pragma unroll
            for (int j = k >> 1; j > 0; j >>= 1) {
                const int32_t y = __shfl_xor_sync(0xffffffffu, x, j);
                const bool up = ((lane & k) == 0) == ((lane & j) == 0);   // this lane keeps the smaller of the pair
                x = up ? min(x, y) : max(x, y);
            }
        if (lane < cnt) v[lane] = x;
        return;
    }
    if (cnt <= PAIR_RANK_MAX) {
        // up to 512: rank sort through shared memory (segment ids are distinct: the rank of an id is the number of smaller
        // ones; n^2 / 32 comparisons per lane on broadcast reads beat a bitonic network that works in global memory --
        // a pixel of a full spill holds ~120 segments)
        __shared__ __align__(16) int32_t s_list[4][PAIR_RANK_MAX];
        int32_t *sl = s_list[threadIdx.x >> 5];
        const int cnt4 = (cnt + 3) & ~3;                                // (padded with ids no segment has: never smaller)
        for (int i = lane; i < cnt4; i += 32) sl[i] = i < cnt ? v[i] : INT32_MAX;
        __syncwarp();
        for (int i = lane; i < cnt; i += 32) {
            const int32_t x = sl[i];
            int r = 0;
            for (int j = 0; j < cnt4; j += 4) {                         // one broadcast 16-byte read per four comparisons
                const int4 q = *(const int4 *)(sl + j);
                r += (q.x < x ? 1 : 0) + (q.y < x ? 1 : 0) + (q.z < x ? 1 : 0) + (q.w < x ? 1 : 0);
            }
            v[r] = x;
        }
        return;
    }
    // longer lists: the same-direction bitonic network on the list in place (first step of every merge pairs i with
    // its mirror image inside the block, so elements past the end behave as +infinity and are simply skipped)
    int P = 64;
    while (P < cnt) P <<= 1;
    for (int k = 2; k <= P; k <<= 1)
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = lane; t < P / 2; t += 32) {
                int i, l;
                if (j == (k >> 1)) {                                   // mirror step
                    const int blk = t / j, off = t - blk * j;
                    i = blk * k + off;  l = blk * k + k - 1 - off;
                } else {
                    const int blk = t / j, off = t - blk * j;
                    i = blk * 2 * j + off;  l = i + j;
                }
                if (l < cnt) {
                    const int32_t a = v[i], b = v[l];
                    if (a > b) { v[i] = b; v[l] = a; }
                }
            }
            __syncwarp();
        }
}

// one thread per charged-pixel grid cell: emit its tiles (one per window that holds charge) and mark the pixels
// they can reach
__global__ void __launch_bounds__(256)
tile_emit_kernel(DevParams p, const DevTpc *__restrict__ tpcs, int64_t cp0, int64_t n_cp, const int32_t *__restrict__ pix_tile0,
                 const unsigned long long *__restrict__ pix_mask, const int32_t *__restrict__ pix_jmin,
                 const int32_t *__restrict__ pix_start, const int32_t *__restrict__ pix_count,
                 int32_t *tile_cp, TileDesc *tile_desc, int2 *tile_list, int64_t tile_cap, int32_t *cell_list,
                 int32_t *act_first, int32_t *act_last, long long *counters)
{
    int64_t cp = cp0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;   // cells [cp0, cp0 + n_cp) of the planned TPCs
    if (cp >= cp0 + n_cp) return;
    unsigned long long mask[MASK_WORDS];
    bool any = false;
#pragma unroll
    for (int wd = 0; wd < MASK_WORDS; ++wd) { mask[wd] = pix_mask[(size_t)cp * MASK_WORDS + wd]; any |= mask[wd] != 0; }
    if (!any) return;
    {
        // the cells that hold tiles, for the per-cell passes behind the plan's synchronisation (one atomic per warp)
        const unsigned act = __activemask();
        const int lane = threadIdx.x & 31, leader = __ffs(act) - 1;
        long long base = 0;
        if (lane == leader) base = (long long)atomicAdd((unsigned long long *)&counters[CNT_CELLS], (unsigned long long)__popc(act));
        base = __shfl_sync(act, base, leader) + __popc(act & ((1u << lane) - 1u));
        if (base < tile_cap) cell_list[base] = (int32_t)cp;
    }
    const int tpc = tpc_of_cell(tpcs, p.n_tpcs, cp);
    const DevTpc &t = tpcs[tpc];
    int rel = (int)(cp - t.cp_base);
    int px = rel % t.gw - p.H, py = rel / t.gw - p.H;
    int64_t tix = pix_tile0[cp];
    const int js = pix_jmin[cp] & ~3;
    int w_lo = -1, w_hi = -1;
#pragma unroll
    for (int wd = 0; wd < MASK_WORDS; ++wd)
        for (unsigned long long m = mask[wd]; m; m &= m - 1) {
            int w = 64 * wd + __ffsll((long long)m) - 1;
            if (w_lo < 0) w_lo = w;
            w_hi = w;
            if (tix < tile_cap) {
                tile_cp[tix] = (int32_t)cp;
                tile_desc[tix] = TileDesc{tpc, px, py, js + w * p.Jc};
                tile_list[tix] = make_int2(pix_start[cp], pix_count[cp]);
            }
            else atomicAdd((unsigned long long *)&counters[CNT_OVERFLOW], 1ull);
            ++tix;
        }
    int first = js + w_lo * p.Jc;
    int last = min(js + w_hi * p.Jc + p.Jc + p.K - 2, p.n_ticks - 1);
    for (int iy = max(py - p.H, 0); iy <= min(py + p.H, t.ny - 1); ++iy)
        for (int ix = max(px - p.H, 0); ix <= min(px + p.H, t.nx - 1); ++ix) {
            int gp = t.first_pixel_id + iy * t.nx + ix;
            atomicMin(&act_first[gp], first);
            atomicMax(&act_last[gp], last);
        }
}

struct NpixF { const int32_t *v; __device__ long long operator()(int64_t i) const { return v[i]; } };
struct PopcF {
    const unsigned long long *m;
    __device__ long long operator()(int64_t i) const
    {
        int c = 0;
#pragma unroll
        for (int wd = 0; wd < MASK_WORDS; ++wd) c += __popcll(m[(size_t)i * MASK_WORDS + wd]);
        return c;
    }
};
struct ActiveF { const int32_t *last; __device__ long long operator()(int64_t i) const { return last[i] >= 0 ? 1 : 0; } };
struct ActiveLenF {
    const int32_t *first, *last;
    __device__ long long operator()(int64_t i) const { return last[i] >= 0 ? (long long)(last[i] - first[i] + 1) : 0; }
};

// the plan's tables of the cells / pixels of the planned TPCs and its counters, back to "nothing charged" (one launch)
__global__ void __launch_bounds__(256)
plan_reset_kernel(int64_t ncp, int64_t npix, int32_t *pix_count, int32_t *pix_cursor, unsigned long long *pix_mask, int32_t *pix_jmin,
                  int32_t *act_first, int32_t *act_last, long long *counters)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < ncp) {
        pix_count[i] = 0;  pix_cursor[i] = 0;  pix_jmin[i] = INT32_MAX;
#pragma unroll
        for (int wd = 0; wd < MASK_WORDS; ++wd) pix_mask[i * MASK_WORDS + wd] = 0ull;
    }
    if (i < npix) { act_first[i] = INT32_MAX;  act_last[i] = -1; }
    if (i < CNT_COUNT) counters[i] = 0;
}

int sim_ensure_scan_tmp(lartpc_sim *sim, int64_t elems)
{
    int64_t need = lscan::tmp_elems(elems);
    if (need > sim->scan_tmp_elems) {
        if (sim->scan_tmp) cudaFree(sim->scan_tmp);
        sim->scan_tmp = nullptr;
        LARTPC_CUDA_TRY(cudaMalloc(&sim->scan_tmp, sizeof(long long) * need));
        sim->scan_tmp_elems = need;
    }
    return LARTPC_OK;
}


// (re)allocates every per-tile planning array for `cap` tiles
int sim_grow_tiles(lartpc_sim *sim, int64_t cap)
{
    cudaFree(sim->tile_cp); cudaFree(sim->tile_desc); cudaFree(sim->tile_list); cudaFree(sim->tile_perm); cudaFree(sim->cell_list);
    cudaFree(sim->tile_desc_p); cudaFree(sim->tile_list_p); cudaFree(sim->tb_mask); cudaFree(sim->tc_cmask);
    sim->tile_cp = nullptr; sim->tile_desc = nullptr; sim->tile_list = nullptr; sim->tile_perm = nullptr; sim->cell_list = nullptr;
    sim->tile_desc_p = nullptr; sim->tile_list_p = nullptr; sim->tb_mask = nullptr; sim->tc_cmask = nullptr; sim->tile_cap = 0;
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_cp, sizeof(int32_t) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_desc, sizeof(TileDesc) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_list, sizeof(int2) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->cell_list, sizeof(int32_t) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_perm, sizeof(int32_t) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_desc_p, sizeof(TileDesc) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tile_list_p, sizeof(int2) * cap));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tb_mask, sizeof(int32_t) * (cap / TC_TILE_BLOCK + 2)));
    LARTPC_CUDA_TRY(cudaMalloc(&sim->tc_cmask, sizeof(int32_t) * (cap / TC_TILE_BLOCK + 2) * TC_CMASK_WORDS));
    if (!sim->cls_hist) LARTPC_CUDA_TRY(cudaMalloc(&sim->cls_hist, sizeof(int32_t) * (2 * TC_CLASSES + 2)));   // + the own-list cursor
    sim->tile_cap = cap;
    return LARTPC_OK;
}

// ---- tensor-core mode: tiles sorted by the 16-tick arrival blocks and the LUT bins they charge -----------------------
// The response multiplies 128 tiles at a time and can skip a (bin, 16-tick block) pair only when none of the 128 charges
// it (the charge lattice ORs what each tile really charges into a per-unit mask, tc_cmask).  So tiles that charge the
// same blocks AND about the same bins are given neighbouring slots: class = (block mask, box of charged bins with its
// four edges taken in steps of two bins), counting sort over the TC_CLASSES classes in that order; the order inside a
// class is whatever the atomics give: a tile's slot only decides where its rows live, never a sum.  Measured on
// configs[3] / configs[2]: 23 % / 33 % of the (unit, bin, block) pairs drop out (profiles/r2_response_bound.md).

// One warp per charged pixel.  Every tile of the pixel (one per 64-tick window that holds charge) needs the segments of the
// pixel's list that reach its window: they give the tile's class (block mask, box of charged bins), and they are written
// out once more, in the same order, behind the pixels' lists (own_base) as the tile's OWN list -- the charge lattice walks
// a tile's list segment by segment, and a pixel that is hit again and again over a spill (~120 segments at configs[3])
// has ~7 in any one window (charge lattice 100 -> 63 ms).  The lanes read the list 32 segments at a time, once to count
// and classify, once to write; a segment names its windows itself, so the work is linear in the list, not list x tiles.
// Tiles that find no room behind the lists keep the list of their pixel (tile_emit_kernel wrote it).
constexpr int PC_WARPS = 8;
__global__ void __launch_bounds__(32 * PC_WARPS)
pixel_class_kernel(DevParams p, int64_t n_cells, const int32_t *__restrict__ cell_list, const int32_t *__restrict__ pix_start,
                   const int32_t *__restrict__ pix_count, const int32_t *__restrict__ pix_tile0,
                   const unsigned long long *__restrict__ pix_mask, const int32_t *__restrict__ pix_jmin,
                   const TileDesc *__restrict__ td, int2 *tl, int32_t *pair_seg, lartpc_pixmap_t pm,
                   const void *__restrict__ seg_rec, int32_t *cls, int32_t *hist, int64_t own_base, int64_t own_cap)
{
    __shared__ int s_w0[PC_WARPS][MAX_WINDOWS], s_w1[PC_WARPS][MAX_WINDOWS], s_n[PC_WARPS][MAX_WINDOWS];
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    const int64_t ci = (int64_t)blockIdx.x * PC_WARPS + wp;
    if (ci >= n_cells) return;                                        // (warp-uniform, as everything below that returns)
    const int64_t cp = cell_list[ci];
    const unsigned long long m0 = pix_mask[(size_t)cp * MASK_WORDS], m1 = pix_mask[(size_t)cp * MASK_WORDS + 1];
    static_assert(MASK_WORDS == 2, "two 64-bit window words per charged pixel");
    const int cnt = pix_count[cp];
    if ((m0 | m1) == 0ull) return;
    const int nt = __popcll(m0) + __popcll(m1);
    const int64_t tile0 = pix_tile0[cp];
    if (cnt <= 0) {                                                   // (a window bit without a segment: not produced by the plan)
        for (int r = lane; r < nt; r += 32) cls[tile0 + r] = 0;
        return;
    }
    const int start = pix_start[cp];
    const TileDesc d0 = td[tile0];
    const int A_t = d0.px * p.nb, B_t = d0.py * p.nb, js = pix_jmin[cp] & ~3;   // window w starts at tick js + w Jc (tile_emit_kernel)
    int *w0s = s_w0[wp], *w1s = s_w1[wp], *ns = s_n[wp];
    for (int r = lane; r < nt; r += 32) { w0s[r] = 0;  w1s[r] = 0;  ns[r] = 0; }
    __syncwarp();
    // the bits of a mask word (windows base .. base + 63) that lie in windows [lo, hi]
    auto clip = [](unsigned long long m, int base, int lo, int hi) {
        lo -= base;  hi -= base;
        if (hi < 0 || lo > 63) return 0ull;
        if (lo > 0) m &= ~0ull << lo;
        if (hi < 63) m &= (2ull << hi) - 1ull;
        return m;
    };
    auto rank = [&](int w) { return w < 64 ? __popcll(m0 & ((1ull << w) - 1ull)) : __popcll(m0) + __popcll(m1 & ((1ull << (w - 64)) - 1ull)); };
    auto fdiv = [&](int x) { return x >= 0 ? x / p.Jc : -((-x + p.Jc - 1) / p.Jc); };
    // segment k of the list: its id, the windows [wlo, whi] it reaches, its ticks clamped to the read-out, its bins on this pixel
    auto load = [&](int k, int &sid, int &wlo, int &whi, int &t0, int &t1, int &abits, int &bbits) {
        wlo = MAX_WINDOWS;  whi = -1;  abits = bbits = 0;  t0 = t1 = 0;  sid = 0;
        if (k >= cnt) return;
        const int s = pair_seg[start + k];
        sid = s;
        int s_alo, s_ahi, s_blo, s_bhi, s_jt0, s_jt1;
        if (seg_rec) {
            // one 32-byte sector of its record (SEG_REC_BYTES / SEG_REC_BOX_OFFSET: the eight ints {N, a_lo, a_hi, b_lo |
            // b_hi, jt0, jt1, flags} that end the record seg_record_kernel wrote), not six arrays
            const int4 *r = (const int4 *)((const char *)seg_rec + (size_t)SEG_REC_BYTES * s + SEG_REC_BOX_OFFSET);
            const int4 r0 = __ldg(r), r1 = __ldg(r + 1);
            s_alo = r0.y;  s_ahi = r0.z;  s_blo = r0.w;  s_bhi = r1.x;  s_jt0 = r1.y;  s_jt1 = r1.z;
        } else {
            s_alo = pm.a_lo[s];  s_ahi = pm.a_hi[s];  s_blo = pm.b_lo[s];  s_bhi = pm.b_hi[s];  s_jt0 = pm.jt0[s];  s_jt1 = pm.jt1[s];
        }
        t0 = max(s_jt0, 0);  t1 = min(s_jt1, p.j_max);
        if (t0 > t1) return;                                          // never read out
        wlo = max(fdiv(t0 - js), 0);  whi = min(fdiv(t1 - js), MAX_WINDOWS - 1);
        const int al = max(s_alo - A_t, 0), ah = min(s_ahi - A_t, p.nb - 1), bl = max(s_blo - B_t, 0), bh = min(s_bhi - B_t, p.nb - 1);
        if (al <= ah) abits = ((2 << ah) - 1) & ~((1 << al) - 1);
        if (bl <= bh) bbits = ((2 << bh) - 1) & ~((1 << bl) - 1);
    };
    // pass 1: per tile the 16-tick blocks and bins its segments charge, and how many segments those are
    for (int k0 = 0; k0 < cnt; k0 += 32) {
        int sid, wlo, whi, t0, t1, abits, bbits;
        load(k0 + lane, sid, wlo, whi, t0, t1, abits, bbits);
        const int c_lo = __reduce_min_sync(0xffffffffu, wlo), c_hi = __reduce_max_sync(0xffffffffu, whi);
        for (int wd = 0; wd < MASK_WORDS; ++wd)
        for (unsigned long long mm = clip(wd ? m1 : m0, 64 * wd, c_lo, c_hi); mm; mm &= mm - 1) {   // the pixel's windows in [c_lo, c_hi]
            const int w = 64 * wd + __ffsll((long long)mm) - 1;
            const bool m = wlo <= w && w <= whi;
            const unsigned bal = __ballot_sync(0xffffffffu, m);
            if (!bal) continue;
            int v0 = 0;
            if (m) {
                const int jw = js + w * p.Jc, jlo = max(t0 - jw, 0), jhi = min(t1 - jw, p.Jc - 1);
                v0 = (((2 << (jhi >> 4)) - 1) & ~((1 << (jlo >> 4)) - 1)) | (abits << 4);
            }
            const unsigned o0 = __reduce_or_sync(0xffffffffu, (unsigned)v0), o1 = __reduce_or_sync(0xffffffffu, (unsigned)(m ? bbits : 0));
            if (lane == 0) { const int r = rank(w);  w0s[r] |= (int)o0;  w1s[r] |= (int)o1;  ns[r] += __popc(bal); }
        }
    }
    __syncwarp();
    // classes; where the tiles' own lists start (tiles that take the whole list keep it)
    long long total = 0;
    for (int r0 = 0; r0 < nt; r0 += 32) {
        const int r = r0 + lane;
        int own = 0;
        if (r < nt) {
            const int v0 = w0s[r], v1 = w1s[r], n = ns[r];
            const int mask = v0 & 15, ab = v0 >> 4;
            // edges in TC_BOXQ steps over the pixel (any bins_per_pixel); an empty box sorts first
            const int q = (p.nb + TC_BOXQ - 1) / TC_BOXQ;
            const int e0 = ab ? (__ffs(ab) - 1) / q : 0, e1 = ab ? (31 - __clz(ab)) / q : 0;
            const int e2 = v1 ? (__ffs(v1) - 1) / q : 0, e3 = v1 ? (31 - __clz(v1)) / q : 0;
            cls[tile0 + r] = (((mask * TC_BOXQ + e0) * TC_BOXQ + e1) * TC_BOXQ + e2) * TC_BOXQ + e3;
            own = n < cnt ? n : 0;
        }
        int inc = own;
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (r < nt) w1s[r] = own ? (int)total + inc - own : -1;      // offset inside the pixel's block, -1: keeps the pixel's list
        total += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (total == 0 || own_cap <= 0) return;
    long long base = 0;
    if (lane == 0) base = (long long)atomicAdd((unsigned long long *)(hist + 2 * TC_CLASSES), (unsigned long long)total);
    base = __shfl_sync(0xffffffffu, base, 0);
    if (base + total > own_cap) return;
    __syncwarp();
    for (int r = lane; r < nt; r += 32)
        if (w1s[r] >= 0) tl[tile0 + r] = make_int2((int)(own_base + base + w1s[r]), ns[r]);
    int32_t *dst = pair_seg + own_base + base;
    // pass 2: the same walk, writing (w1s[r]: next free place of tile r)
    for (int k0 = 0; k0 < cnt; k0 += 32) {
        int sid, wlo, whi, t0, t1, abits, bbits;
        load(k0 + lane, sid, wlo, whi, t0, t1, abits, bbits);
        const int c_lo = __reduce_min_sync(0xffffffffu, wlo), c_hi = __reduce_max_sync(0xffffffffu, whi);
        for (int wd = 0; wd < MASK_WORDS; ++wd)
        for (unsigned long long mm = clip(wd ? m1 : m0, 64 * wd, c_lo, c_hi); mm; mm &= mm - 1) {   // the pixel's windows in [c_lo, c_hi]
            const int w = 64 * wd + __ffsll((long long)mm) - 1;
            const bool m = wlo <= w && w <= whi;
            const unsigned bal = __ballot_sync(0xffffffffu, m);
            if (!bal) continue;
            const int r = rank(w), at = w1s[r];
            __syncwarp();
            if (at >= 0) {
                if (m) dst[at + __popc(bal & ((1u << lane) - 1u))] = sid;
                if (lane == 0) w1s[r] = at + __popc(bal);
            }
            __syncwarp();
        }
    }
}

// tiles in their original order (no sort): every block, no box
__global__ void __launch_bounds__(256) tile_class_flat_kernel(int64_t n_tiles, int32_t *cls)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_tiles) cls[t] = 15 * TC_BOX_CLASSES;
}

// class counts: one atomic per (warp, class)
__global__ void __launch_bounds__(256) class_hist_kernel(int64_t n_tiles, const int32_t *__restrict__ cls, int32_t *hist)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int c = t < n_tiles ? cls[t] : TC_CLASSES;                  // no tile: a group of its own
    const int lane = threadIdx.x & 31;
    const unsigned peers = __match_any_sync(0xffffffffu, c);
    if (lane == __ffs(peers) - 1 && c < TC_CLASSES) atomicAdd(&hist[c], __popc(peers));
}

// hist[0 .. TC_CLASSES) counts -> hist[TC_CLASSES .. 2 TC_CLASSES) first slot of the class (one CTA of 1024 threads)
__global__ void __launch_bounds__(1024) class_offsets_kernel(int32_t *hist)
{
    __shared__ int s_part[32];
    constexpr int PER = (TC_CLASSES + 1023) / 1024;
    const int k0 = threadIdx.x * PER;
    int sum = 0;
    for (int k = k0; k < min(k0 + PER, TC_CLASSES); ++k) sum += hist[k];
    // exclusive scan of the 1 024 partial sums: within warps by shuffles, then over the 32 warp totals
    const int lane = threadIdx.x & 31, wp = threadIdx.x >> 5;
    int inc = sum;
    for (int o = 1; o < 32; o <<= 1) {
        const int y = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += y;
    }
    if (lane == 31) s_part[wp] = inc;
    __syncthreads();
    if (wp == 0) {
        const int t = s_part[lane];
        int ti = t;
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, ti, o);
            if (lane >= o) ti += y;
        }
        s_part[lane] = ti - t;
    }
    __syncthreads();
    int run = s_part[wp] + inc - sum;
    for (int k = k0; k < min(k0 + PER, TC_CLASSES); ++k) { hist[TC_CLASSES + k] = run;  run += hist[k]; }
}

__global__ void __launch_bounds__(256)
tile_scatter_kernel(int64_t n_tiles, int32_t *perm /* in: class, out: slot */, int32_t *hist, const TileDesc *__restrict__ td,
                    const int2 *__restrict__ tl, TileDesc *td_p, int2 *tl_p, int32_t *tb_mask, int sort)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = t < n_tiles;
    const int c = valid ? perm[t] : TC_CLASSES;                       // TC_CLASSES: no tile (its own group below)
    int slot = (int)t;
    if (sort) {
        // one atomic per (warp, class): the lanes of a class take consecutive slots
        const int lane = threadIdx.x & 31;
        const unsigned peers = __match_any_sync(0xffffffffu, c);
        const int leader = __ffs(peers) - 1;
        int base = 0;
        if (lane == leader && valid) base = atomicAdd(&hist[TC_CLASSES + c], __popc(peers));
        base = __shfl_sync(0xffffffffu, base, leader);
        slot = base + __popc(peers & ((1u << lane) - 1u));
    }
    if (!valid) return;
    const int mask = c / TC_BOX_CLASSES;
    perm[t] = slot;
    td_p[slot] = td[t];
    tl_p[slot] = tl[t];
    if (mask) atomicOr(&tb_mask[slot / TC_UNIT_TILES], mask);
}

static int grow_i32(int32_t **p, int64_t *cap, int64_t need)
{
    if (need <= *cap) return LARTPC_OK;
    if (*p) cudaFree(*p);
    *p = nullptr;
    int64_t c = need + need / 4 + 1024;
    LARTPC_CUDA_TRY(cudaMalloc(p, sizeof(int32_t) * c));
    *cap = c;
    return LARTPC_OK;
}

// the same, keeping the first `keep` elements (the copy is ordered behind what wrote them on `st`)
static int grow_i32_keep(int32_t **p, int64_t *cap, int64_t need, int64_t keep, cudaStream_t st)
{
    if (need <= *cap) return LARTPC_OK;
    int32_t *q = nullptr;
    const int64_t c = need + need / 8 + 1024;
    LARTPC_CUDA_TRY(cudaMalloc(&q, sizeof(int32_t) * c));
    if (*p && keep > 0) LARTPC_CUDA_TRY(cudaMemcpyAsync(q, *p, sizeof(int32_t) * keep, cudaMemcpyDeviceToDevice, st));
    LARTPC_CUDA_TRY(cudaStreamSynchronize(st));
    if (*p) cudaFree(*p);
    *p = q;
    *cap = c;
    return LARTPC_OK;
}

// S3 launcher.  Segments whose TPC lies outside [tpc_lo, tpc_hi) get their rectangles but no tiles
// (lartpc_run_spill plans one TPC batch at a time; the staged API passes the full range).
int launch_plan(lartpc_sim *sim, const lartpc_segments_t *seg, const lartpc_drifted_t *dr, int64_t n,
                int tpc_lo, int tpc_hi, lartpc_pixmap_t *out, lartpc_pixmap_info_t *info, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    SegPtrs s{seg->xs, seg->ys, seg->zs, seg->ts, seg->xe, seg->ye, seg->ze, seg->te, seg->dE};
    int rc;
    if ((rc = sim_ensure_scan_tmp(sim, sim->n_cp > n ? sim->n_cp : (n > sim->n_pix ? n : sim->n_pix))) != 0) return rc;
    sim->have_plan = false;
    sim->have_signals = false;
    if (tpc_lo < 0 || tpc_hi > p.n_tpcs || tpc_lo > tpc_hi) return LARTPC_ERR_BAD_ARGUMENT;
    const int64_t cp_lo = sim->cp_base_h[tpc_lo], ncp = sim->cp_base_h[tpc_hi] - cp_lo;
    const int64_t pix_lo = sim->pix_base_h[tpc_lo], npix = sim->pix_base_h[tpc_hi] - pix_lo;
    sim->plan_pix_lo = pix_lo;  sim->plan_pix_hi = pix_lo + npix;
    // a later TPC batch of the input whose boxes the tpc_lo = 0 plan wrote into these very arrays (lartpc_run_spill)
    const int reuse = (tpc_lo > 0 && sim->boxes_n == n && sim->boxes_of == (const void *)out->a_lo && n > 0) ? 1 : 0;
    if (tpc_lo == 0) { sim->boxes_n = -1;  sim->boxes_of = nullptr; }

    for (int attempt = 0; attempt < 2; ++attempt) {
        // only the cells and pixels of the planned TPCs are touched (lartpc_run_spill plans a few TPCs at a time)
        ++g_lartpc_launches;
        plan_reset_kernel<<<div_up(std::max<int64_t>(std::max(ncp, npix), CNT_COUNT), 256), 256, 0, st>>>(
            ncp, npix, sim->pix_count + cp_lo, sim->pix_cursor + cp_lo, sim->pix_mask + cp_lo * MASK_WORDS, sim->pix_jmin + cp_lo,
            sim->act_first + pix_lo, sim->act_last + pix_lo, sim->d_counters);
        if (n > 0) {
            ++g_lartpc_launches;
            pixmap_kernel<<<div_up(n, 256), 256, 0, st>>>(p, sim->d_tpcs, s, n, dr->tpc, dr->q_anode, tpc_lo, tpc_hi,
                                                         *out, sim->pix_count, sim->pix_jmin, sim->d_counters, reuse);
            LARTPC_CUDA_TRY(cudaGetLastError());
        }
        // per-segment records of the tensor-core splat: once per plan of the whole input
        if (tpc_lo == 0 && (rc = launch_seg_records(sim, dr, out, n, st)) != 0) return rc;
        // offsets[n+1] = exclusive scan of npix
        if (!reuse)
            LARTPC_CUDA_TRY(lscan::exclusive_scan(n, NpixF{out->npix}, out->offsets, true,
                                                  sim->d_counters + CNT_TOTAL_NPIX, sim->scan_tmp, st));
        // per charged pixel: start of its segment list
        LARTPC_CUDA_TRY(lscan::exclusive_scan(ncp, NpixF{sim->pix_count + cp_lo}, sim->pix_start + cp_lo, false,
                                              (long long *)nullptr, sim->scan_tmp, st));
        if (n > 0) {
            ++g_lartpc_launches;
            pair_fill_kernel<<<div_up(n, 256), 256, 0, st>>>(p, sim->d_tpcs, n, dr->tpc, *out, tpc_lo, tpc_hi,
                                                            sim->pix_start, sim->pix_cursor, sim->pix_jmin,
                                                            sim->pix_mask, sim->pair_seg, sim->pair_cap,
                                                            sim->d_counters);
        }
        // index of the first tile of every charged pixel (one tile per window that holds charge)
        LARTPC_CUDA_TRY(lscan::exclusive_scan(ncp, PopcF{sim->pix_mask + cp_lo * MASK_WORDS}, sim->pix_tile0 + cp_lo, false,
                                              sim->d_counters + CNT_TILES, sim->scan_tmp, st));
        ++g_lartpc_launches;
        tile_emit_kernel<<<div_up(ncp, 256), 256, 0, st>>>(p, sim->d_tpcs, cp_lo, ncp, sim->pix_tile0,
                                                                sim->pix_mask, sim->pix_jmin, sim->pix_start,
                                                                sim->pix_count, sim->tile_cp, sim->tile_desc,
                                                                sim->tile_list, sim->tile_cap, sim->cell_list,
                                                                sim->act_first, sim->act_last, sim->d_counters);
        LARTPC_CUDA_TRY(cudaGetLastError());
        // active pixels: slot = rank among active pixels (sorted by id), total waveform samples
        LARTPC_CUDA_TRY(lscan::exclusive_scan(npix, ActiveF{sim->act_last + pix_lo}, sim->act_slot + pix_lo, false,
                                              sim->d_counters + CNT_ACTIVE_PIX, sim->scan_tmp, st));
        LARTPC_CUDA_TRY(lscan::exclusive_scan(npix, ActiveLenF{sim->act_first + pix_lo, sim->act_last + pix_lo},
                                              (long long *)nullptr, false, sim->d_counters + CNT_TOTAL_SAMPLES,
                                              sim->scan_tmp, st));
        LARTPC_CUDA_TRY(cudaMemcpyAsync(sim->h_counters, sim->d_counters, sizeof(long long) * CNT_COUNT,
                                        cudaMemcpyDeviceToHost, st));
        LARTPC_CUDA_TRY(cudaStreamSynchronize(st));
        const long long *h = sim->h_counters;
        if (h[CNT_OVERFLOW] == 0) break;
        if (attempt == 1) return LARTPC_ERR_CAPACITY;
        // grow the plan buffers to the sizes just counted and plan again
        if ((rc = grow_i32(&sim->pair_seg, &sim->pair_cap, h[CNT_PAIRS])) != 0) return rc;
        if (h[CNT_TILES] > sim->tile_cap && (rc = sim_grow_tiles(sim, h[CNT_TILES] + h[CNT_TILES] / 4 + 1024)) != 0) return rc;
    }
    const long long *h = sim->h_counters;
    sim->plan_n = n;
    sim->n_tiles = h[CNT_TILES];
    const int64_t n_cells = h[CNT_CELLS];
    if (n_cells > 0) {
        // the atomics of pair_fill_kernel fill each list in arbitrary order: sort it by segment id (one warp per cell)
        ++g_lartpc_launches;
        pair_sort_kernel<<<div_up(n_cells, 4), 128, 0, st>>>(n_cells, sim->cell_list, sim->pix_start, sim->pix_count,
                                                              sim->pair_seg, sim->pair_cap);
    }
    if (tpc_lo == 0) { sim->need_composite = h[CNT_COMPOSITE] != 0;  sim->boxes_n = n;  sim->boxes_of = (const void *)out->a_lo; }
    if (p.tc_mode && sim->n_tiles > 0) {
        // the FFMA2 splat (bins per pixel other than 5 / 10) writes the operand image in the tiles' original order
        const int sort = splat_on_tc(p) ? 1 : 0;
        const int64_t nt = sim->n_tiles;
        LARTPC_CUDA_TRY(cudaMemsetAsync(sim->cls_hist, 0, sizeof(int32_t) * (2 * TC_CLASSES + 2), st));
        // room behind the pixels' lists for the tiles' own lists: a segment charges one or two windows of a pixel
        int64_t own_cap = 0;
        if (sort && h[CNT_PAIRS] > 0) {
            own_cap = std::min<int64_t>(2 * h[CNT_PAIRS] + 4096, (int64_t)INT32_MAX - h[CNT_PAIRS] - 1);
            if ((rc = grow_i32_keep(&sim->pair_seg, &sim->pair_cap, h[CNT_PAIRS] + own_cap, h[CNT_PAIRS], st)) != 0) return rc;
        }
        LARTPC_CUDA_TRY(cudaMemsetAsync(sim->tb_mask, 0, sizeof(int32_t) * (nt / TC_TILE_BLOCK + 1), st));
        g_lartpc_launches += 4;
        if (sort)
            pixel_class_kernel<<<div_up(n_cells, PC_WARPS), 32 * PC_WARPS, 0, st>>>(
                p, n_cells, sim->cell_list, sim->pix_start, sim->pix_count, sim->pix_tile0, sim->pix_mask, sim->pix_jmin, sim->tile_desc,
                sim->tile_list, sim->pair_seg, *out, sim->seg_rec_cap >= n ? sim->seg_rec : nullptr, sim->tile_perm,
                sim->cls_hist, h[CNT_PAIRS], own_cap);
        else tile_class_flat_kernel<<<div_up(nt, 256), 256, 0, st>>>(nt, sim->tile_perm);
        class_hist_kernel<<<div_up(nt, 256), 256, 0, st>>>(nt, sim->tile_perm, sim->cls_hist);
        class_offsets_kernel<<<1, 1024, 0, st>>>(sim->cls_hist);
        tile_scatter_kernel<<<div_up(nt, 256), 256, 0, st>>>(nt, sim->tile_perm, sim->cls_hist, sim->tile_desc,
                                                            sim->tile_list, sim->tile_desc_p, sim->tile_list_p,
                                                            sim->tb_mask, sort);
        LARTPC_CUDA_TRY(cudaGetLastError());
    }
    sim->n_pairs = h[CNT_PAIRS];
    sim->n_active = h[CNT_ACTIVE_PIX];
    sim->total_samples = h[CNT_TOTAL_SAMPLES];
    sim->drifted_copy = *dr;
    sim->pixmap_copy = *out;
    sim->have_plan = true;
    if (info) {
        info->max_npix = (int32_t)h[CNT_MAX_NPIX];
        info->max_ticks = (int32_t)h[CNT_MAX_TICKS];
        info->total_npix = h[CNT_TOTAL_NPIX];
        info->n_active_segments = h[CNT_ACTIVE_SEGS];
        info->n_tiles = h[CNT_TILES];
        info->n_pairs = h[CNT_PAIRS];
        info->n_active_pixels = h[CNT_ACTIVE_PIX];
        info->total_samples = h[CNT_TOTAL_SAMPLES];
        info->tile_targets = p.WW * p.nq;                               // rows of `partial` per tile
        info->tile_ticks = p.tile_ticks;
        info->tile_charge_floats = p.slab_floats;
        info->tile_block = p.tc_mode ? TC_UNIT_TILES : 1;
    }
    return LARTPC_OK;
}
