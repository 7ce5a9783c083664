// S5 per-pixel sum and S6 LArPix-style electronics: parallel over pixels.
#include "common.cuh"
#include "scan.cuh"

// -------------------------------------------------------------------------------------------------
// S5: active-pixel table (sorted by pixel id) and the gather-sum of the tile partial waveforms.
// Every sample is written once by one thread, adding the <= W*W x 3 contributing tiles in a fixed
// order (target index ascending, chunk ascending), so the sum is reproducible bit for bit.
// -------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
active_table_kernel(int64_t pix0, int64_t n_pix, const int32_t *__restrict__ act_first, const int32_t *__restrict__ act_last,
                    const int32_t *__restrict__ act_slot, int32_t *pixel_id, int32_t *first_tick, int32_t *length)
{
    int64_t gp = pix0 + (int64_t)blockIdx.x * blockDim.x + threadIdx.x;    // pixels of the planned TPCs
    if (gp >= pix0 + n_pix) return;
    int last = act_last[gp];
    if (last < 0) return;
    int slot = act_slot[gp];
    pixel_id[slot] = (int32_t)gp;
    first_tick[slot] = act_first[gp];
    length[slot] = last - act_first[gp] + 1;
}

struct LenF { const int32_t *v; __device__ long long operator()(int64_t i) const { return v[i]; } };

#ifndef LARTPC_SUM_MLP
#define LARTPC_SUM_MLP 4
#endif
constexpr int SUM_MLP = LARTPC_SUM_MLP;   // listed rows a thread loads before it adds them (in list order); measured at configs[3]: 4 -> 21.5 ms, 6 -> 22.0, 8 -> 24.4
constexpr int SUM_THREADS = 128;
constexpr int SUM_LCAP = 448;      // partial rows listed per round (W*W x the charge windows of the pixels around: ~30 on a lone track, ~200 in a full spill)

// CTA = active pixel.  Its threads first list, one row each and all at once, the partial rows that reach the pixel: for target
// index d of the W x W window and every charge window of that charged pixel (d ascending, window ascending), the row of the
// tile (through the slot map) and the ticks it can be non-zero on.  Then a thread owns VEC consecutive ticks of the waveform
// and adds the listed rows in list order: the order of the float32 additions -- hence every output bit -- is fixed.
template <int VEC, bool PIECES>    // VEC: ticks per thread and load, 4 when tile_ticks is a multiple of 4 (rows 16-byte aligned), else 2
                                   // PIECES: a long LUT cut into pieces (tensor-core path, K > 209): nq rows per (tile, target)
__global__ void __launch_bounds__(SUM_THREADS)
sum_pixel_kernel(DevParams p, const DevTpc *__restrict__ tpcs, const int32_t *__restrict__ pixel_id,
                 const int32_t *__restrict__ first_tick, const int32_t *__restrict__ length,
                 const int64_t *__restrict__ offset, const unsigned long long *__restrict__ pix_mask,
                 const int32_t *__restrict__ pix_tile0, const int32_t *__restrict__ pix_jmin,
                 const float *__restrict__ partial, const int32_t *__restrict__ tile_range,
                 const int32_t *__restrict__ tile_perm /* slot of a tile, or null: identity */, float *samples)
{
    __shared__ unsigned long long s_mask[128][MASK_WORDS];
    __shared__ int s_tile0[128], s_js[128], s_base[129];
    __shared__ const float *e_row[SUM_LCAP];
    __shared__ int e_na[SUM_LCAP], e_nb[SUM_LCAP];
    const int slot = blockIdx.x, tid = threadIdx.x;
    const int gp = pixel_id[slot];
    const int tpc = tpc_of_pixel(tpcs, p.n_tpcs, gp);
    const DevTpc &t = tpcs[tpc];
    const int rel = gp - t.first_pixel_id, iy = rel / t.nx, ix = rel - iy * t.nx;
    const int first = first_tick[slot], len = length[slot], last = first + len - 1;
    if (tid < p.WW) {
        const int d = tid, dyi = d / p.W, dxi = d - dyi * p.W;
        const int cp = t.cp_base + (iy + dyi) * t.gw + (ix + dxi);   // charged pixel px = ix - H + dxi
        int cnt = 0;
#pragma unroll
        for (int wd = 0; wd < MASK_WORDS; ++wd) {
            s_mask[d][wd] = pix_mask[(size_t)cp * MASK_WORDS + wd];
            cnt += __popcll(s_mask[d][wd]);
        }
        s_tile0[d] = pix_tile0[cp];
        s_js[d] = pix_jmin[cp] & ~3;                                 // window origin of that charged pixel
        s_base[d + 1] = cnt;
    }
    __syncthreads();
    if (tid == 0) {
        s_base[0] = 0;
        for (int d = 0; d < p.WW; ++d) s_base[d + 1] += s_base[d];
    }
    __syncthreads();
    const int nq = PIECES ? p.nq : 1;                                 // rows per (tile, target): pieces of a long LUT
    const int total = s_base[p.WW] * nq;
    const int64_t off = offset[slot];
    for (int r0 = 0; r0 < total; r0 += SUM_LCAP) {
        // one thread per listed row (all of them at once: the row's tile and tick range are two dependent gathers)
        for (int g = tid; g < min(SUM_LCAP, total - r0); g += SUM_THREADS) {
            const int pr = (g + r0) / nq, q = (g + r0) - pr * nq;     // (target, window) pair of the pixel; piece of a long LUT
            int d = 0;                                                // its target: the last d with s_base[d] <= pr
            for (int step = 64; step; step >>= 1)
                if (d + step < p.WW && s_base[d + step] <= pr) d += step;
            int r = pr - s_base[d];                                   // ... and window: the r-th set bit of that pixel's mask
            const int tix = s_tile0[d] + r;
            unsigned long long m = s_mask[d][0];
            int wbase = 0;
            static_assert(MASK_WORDS == 2, "two 64-bit window words per charged pixel");
            if (r >= __popcll(m)) { r -= __popcll(m);  m = s_mask[d][1];  wbase = 64; }
            for (int i = 0; i < r; ++i) m &= m - 1;
            const int w = wbase + __ffsll((long long)m) - 1;
            const int ts = tile_perm ? tile_perm[tix] : tix;
            const int2 rg = *(const int2 *)(tile_range + TILE_META * ts);       // first / last output block
            const int j_start = s_js[d] + w * p.Jc;
            const int t0 = PIECES ? p.KQ * q : 0;                                // piece q answers KQ q ticks later
            const int lo = max(rg.x * RESP_NO, t0), hi = min(rg.y * RESP_NO + RESP_NO - 1, t0 + p.tile_ticks - 1);
            e_row[g] = partial + (((size_t)ts * p.WW + d) * nq + q) * p.tile_ticks - (j_start + t0);
            e_na[g] = (rg.x > rg.y || lo > hi) ? INT_MAX : max(first, j_start + lo);
            e_nb[g] = (rg.x > rg.y || lo > hi) ? -1 : min(last, j_start + hi);
        }
        __syncthreads();
        const int ne = min(SUM_LCAP, total - r0);
        // a thread owns VEC consecutive ticks starting at a multiple of VEC: window origins are multiples of 4, so that is
        // one aligned load of a row.  A warp owns 32 VEC consecutive ticks: its lanes first find, 32 listed rows at a time,
        // the rows that reach that span at all (a pixel of a full spill lists ~200 rows, a span meets ~50 of them), then
        // walk those four at a time -- four independent loads in flight per thread, added in list order.
        const int n_al0 = first & ~(VEC - 1), lane = tid & 31;
        for (int iv0 = tid & ~31; VEC * iv0 < last - n_al0 + 1; iv0 += SUM_THREADS) {   // (warp-uniform)
            const int n = n_al0 + VEC * (iv0 + lane);
            const int w_lo = n_al0 + VEC * iv0, w_hi = w_lo + 32 * VEC - 1;
            const bool mine = n <= last;
            float a[VEC];
#pragma unroll
            for (int k = 0; k < VEC; ++k) a[k] = (r0 && n + k >= first && n + k <= last) ? samples[off + (n + k - first)] : 0.f;
            for (int e0 = 0; e0 < ne; e0 += 32) {
                const int e = e0 + lane;
                unsigned bal = __ballot_sync(0xffffffffu, e < ne && e_nb[e] >= w_lo && e_na[e] <= w_hi);
                while (bal) {
                    float v[SUM_MLP][VEC];
                    int na[SUM_MLP], nb[SUM_MLP];
#pragma unroll
                    for (int i = 0; i < SUM_MLP; ++i) {
                        na[i] = INT_MAX;  nb[i] = -1;
#pragma unroll
                        for (int k = 0; k < VEC; ++k) v[i][k] = 0.f;
                        if (bal) {
                            const int x = e0 + __ffs(bal) - 1;
                            bal &= bal - 1;
                            const int xa = e_na[x], xb = e_nb[x];
                            if (mine && n + VEC - 1 >= xa && n <= xb) {
                                na[i] = xa;  nb[i] = xb;
                                if (VEC == 4) { const float4 q = __ldcs((const float4 *)(e_row[x] + n)); v[i][0] = q.x; v[i][1] = q.y; v[i][2] = q.z; v[i][3] = q.w; }
                                else { const float2 q = __ldcs((const float2 *)(e_row[x] + n)); v[i][0] = q.x; v[i][1] = q.y; }
                            }
                        }
                    }
#pragma unroll
                    for (int i = 0; i < SUM_MLP; ++i)
#pragma unroll
                        for (int k = 0; k < VEC; ++k)
                            if (n + k >= na[i] && n + k <= nb[i]) a[k] += v[i][k];
                }
            }
            if (mine) {
#pragma unroll
                for (int k = 0; k < VEC; ++k)
                    if (n + k >= first && n + k <= last) samples[off + (n + k - first)] = a[k];
            }
        }
        __syncthreads();
    }
    if (total == 0)
        for (int i = tid; i < len; i += SUM_THREADS) samples[off + i] = 0.f;
}

int launch_sum(lartpc_sim *sim, const lartpc_signals_t *sig, lartpc_waveforms_t *out, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    out->n_active = sim->n_active;
    out->total_samples = sim->total_samples;
    if (sim->n_active == 0) {
        LARTPC_CUDA_TRY(cudaMemsetAsync(out->offset, 0, sizeof(int64_t), st));
        return LARTPC_OK;
    }
    if (p.WW > 128) return LARTPC_ERR_UNSUPPORTED;
    ++g_lartpc_launches;
    active_table_kernel<<<div_up(sim->plan_pix_hi - sim->plan_pix_lo, 256), 256, 0, st>>>(
        sim->plan_pix_lo, sim->plan_pix_hi - sim->plan_pix_lo, sim->act_first, sim->act_last,
                                                                sim->act_slot, out->pixel_id, out->first_tick,
                                                                out->length);
    int rc = sim_ensure_scan_tmp(sim, sim->n_active);
    if (rc) return rc;
    LARTPC_CUDA_TRY(lscan::exclusive_scan(sim->n_active, LenF{out->length}, out->offset, true, (long long *)nullptr,
                                          sim->scan_tmp, st));
    ++g_lartpc_launches;
#define LARTPC_SUM_LAUNCH(V, P) sum_pixel_kernel<V, P><<<(unsigned)sim->n_active, SUM_THREADS, 0, st>>>( \
        p, sim->d_tpcs, out->pixel_id, out->first_tick, out->length, out->offset, sim->pix_mask, sim->pix_tile0, \
        sim->pix_jmin, sig->partial, sig->tile_range, p.tc_mode ? sim->tile_perm : nullptr, out->samples)
    if (p.tc_mode && p.nq > 1) LARTPC_SUM_LAUNCH(4, true);             // (tile_ticks = 264 there)
    else if (p.tile_ticks % 4 == 0) LARTPC_SUM_LAUNCH(4, false);
    else LARTPC_SUM_LAUNCH(2, false);
#undef LARTPC_SUM_LAUNCH
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

// -------------------------------------------------------------------------------------------------
// S6: one thread per active pixel, serial over ticks, state in registers.
// Noise: Philox4x32-10, counter (pixel id, tick, 0, 0), key (seed lo, seed hi); Box-Muller in float64 so
// that the ADC decision is taken in the same precision as the oracle's.
// -------------------------------------------------------------------------------------------------
__device__ __forceinline__ void noise_normals(unsigned long long seed, uint32_t pixel, uint32_t tick, double (&z)[3])
{
    uint32_t x[4];
    philox4x32_10(pixel, tick, 0u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
    const double s = 1.0 / 4294967296.0, two_pi = 6.283185307179586476925286766559;
    const double u0 = ((double)x[0] + 0.5) * s, u1 = ((double)x[1] + 0.5) * s;
    const double u2 = ((double)x[2] + 0.5) * s, u3 = ((double)x[3] + 0.5) * s;
    const double r01 = sqrt(-2.0 * log(u0)), r23 = sqrt(-2.0 * log(u2));
    z[0] = r01 * cos(two_pi * u1);
    z[1] = r01 * sin(two_pi * u1);
    z[2] = r23 * cos(two_pi * u3);
}

constexpr int ADC_SHIFT = 12;   // hit slot = tick << 12 | adc

__global__ void __launch_bounds__(128)
electronics_kernel(DevParams p, unsigned long long seed, int64_t n_active, const int32_t *__restrict__ pixel_id,
                   const int32_t *__restrict__ first_tick, const int32_t *__restrict__ length,
                   const int64_t *__restrict__ offset, const float *__restrict__ samples,
                   const uint32_t *__restrict__ disabled, int32_t *slots, int32_t *hits_per_pixel, float *q_pixel)
{
    const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= n_active) return;
    const int pid = pixel_id[slot];
    const int first = first_tick[slot], len = length[slot];
    const float *w = samples + offset[slot];
    const bool every_tick = p.noise_disc != 0.0 || p.periodic > 0;     // the state can change outside the support
    const bool any_noise = p.noise_disc != 0.0 || p.noise_uncorr != 0.0 || p.noise_reset != 0.0;
    const bool off_channel = disabled && ((disabled[pid >> 5] >> (pid & 31)) & 1u);
    int n_begin = every_tick ? 0 : first;
    int n_end = every_tick ? p.n_ticks : first + len;                    // exclusive; extended while a hold is pending
    double q = 0.0, qsum = 0.0;
    bool armed = true;
    int n_c = 0, nhits = 0;
    long long rearm_at = 0;
    int32_t *my = slots + slot * p.max_hits;
    for (int n = n_begin; n < p.n_ticks; ++n) {
        if (n >= n_end && armed && q < p.threshold) break;            // nothing can happen any more
        double z[3] = {0.0, 0.0, 0.0};
        bool have_z = false;
        if (p.noise_disc != 0.0) { noise_normals(seed, (uint32_t)pid, (uint32_t)n, z); have_z = true; }
        if (armed && p.periodic > 0 && n > 0 && (n % p.periodic) == 0) q = 0.0;
        const int i = n - first;
        const double cur = (i >= 0 && i < len) ? (double)w[i] : 0.0;
        q += cur;  qsum += cur;
        if (armed && n >= rearm_at && q >= p.threshold + p.noise_disc * z[0]) { armed = false; n_c = n; }
        if (!armed && n == n_c + p.hold) {
            if (!have_z && any_noise) noise_normals(seed, (uint32_t)pid, (uint32_t)n, z);
            const double q_s = q + p.noise_uncorr * z[1];
            const double V = p.v_ped + p.gain_mv_per_ke * q_s / 1000.0;
            double a = floor((V - p.v_cm) / (p.v_ref - p.v_cm) * p.adc_full);
            a = fmin(fmax(a, 0.0), p.adc_full - 1.0);
            if (!off_channel) {
                if (nhits < p.max_hits) my[nhits] = (n << ADC_SHIFT) | (int)a;
                ++nhits;
            }
            q = p.noise_reset * z[2];
            armed = true;
            rearm_at = max((long long)n + 1, (long long)n + p.min_spacing - p.hold);
        }
    }
    hits_per_pixel[slot] = nhits;
    q_pixel[slot] = (float)qsum;
}

// Warp per active pixel, for parameter sets whose state can only change on the pixel's own support (no discriminator
// noise, no periodic reset: every BASELINE config).  Same state machine as electronics_kernel, but the charge
// integral runs 32 ticks at a time: lane l holds tick n + l, an inclusive warp scan in float64 gives q after every tick of
// the chunk, the first threshold crossing is a ballot, and the sample / reset 16 ticks later restarts the chunk behind it.
// The loads are coalesced and the serial depth is (support / 32 + 2 per hit) steps instead of one step per tick.
__global__ void __launch_bounds__(128)
electronics_warp_kernel(DevParams p, unsigned long long seed, int64_t n_active, const int32_t *__restrict__ pixel_id,
                        const int32_t *__restrict__ first_tick, const int32_t *__restrict__ length,
                        const int64_t *__restrict__ offset, const float *__restrict__ samples,
                        const uint32_t *__restrict__ disabled, int32_t *slots, int32_t *hits_per_pixel, float *q_pixel)
{
    const int64_t slot = (int64_t)blockIdx.x * (blockDim.x / 32) + (threadIdx.x >> 5);
    if (slot >= n_active) return;
    const int lane = threadIdx.x & 31;
    const int pid = pixel_id[slot];
    const int first = first_tick[slot], len = length[slot];
    const float *w = samples + offset[slot];
    const bool any_noise = p.noise_uncorr != 0.0 || p.noise_reset != 0.0;
    const bool off_channel = disabled && ((disabled[pid >> 5] >> (pid & 31)) & 1u);
    // Q_p = sum of the waveform
    double qsum = 0.0;
    for (int i = lane; i < len; i += 32) qsum += (double)w[i];
    for (int d = 16; d; d >>= 1) qsum += __shfl_xor_sync(0xffffffffu, qsum, d);
    const int n_end = first + len;                                    // exclusive end of the support
    double q = 0.0;
    bool armed = true;
    int n_c = 0, nhits = 0;
    long long rearm_at = 0;
    int32_t *my = slots + slot * p.max_hits;
    int n = first;
    while (n < p.n_ticks) {
        if (n >= n_end && armed && q < p.threshold) break;            // nothing can happen any more
        const int i = n + lane - first;
        const double cur = (i >= 0 && i < len && n + lane < p.n_ticks) ? (double)w[i] : 0.0;
        double pref = cur;                                            // q after tick n + lane, minus q before the chunk
        for (int d = 1; d < 32; d <<= 1) {
            const double o = __shfl_up_sync(0xffffffffu, pref, d);
            if (lane >= d) pref += o;
        }
        pref += q;
        if (armed) {
            const unsigned hit = __ballot_sync(0xffffffffu, (long long)n + lane >= rearm_at && pref >= p.threshold &&
                                                               n + lane < p.n_ticks);
            if (hit) { armed = false; n_c = n + __ffs(hit) - 1; }
        }
        if (!armed) {
            const int ns = n_c + p.hold;                              // digitisation tick (D14)
            if (ns >= p.n_ticks) break;                               // the sample falls past the window: no hit
            if (ns <= n + 31) {
                const double q_at = __shfl_sync(0xffffffffu, pref, ns - n);
                double z[3] = {0.0, 0.0, 0.0};
                if (any_noise) noise_normals(seed, (uint32_t)pid, (uint32_t)ns, z);
                const double q_s = q_at + p.noise_uncorr * z[1];
                const double V = p.v_ped + p.gain_mv_per_ke * q_s / 1000.0;
                double a = floor((V - p.v_cm) / (p.v_ref - p.v_cm) * p.adc_full);
                a = fmin(fmax(a, 0.0), p.adc_full - 1.0);
                if (!off_channel) {
                    if (nhits < p.max_hits && lane == 0) my[nhits] = (ns << ADC_SHIFT) | (int)a;
                    ++nhits;
                }
                q = p.noise_reset * z[2];
                armed = true;
                rearm_at = max((long long)ns + 1, (long long)ns + p.min_spacing - p.hold);
                n = ns + 1;                                           // the ticks behind the sample start from the new q
                continue;
            }
        }
        q = __shfl_sync(0xffffffffu, pref, 31);
        n += 32;
    }
    if (lane == 0) {
        hits_per_pixel[slot] = nhits;
        q_pixel[slot] = (float)qsum;
    }
}

struct HitCountF {
    const int32_t *v; int cap;
    __device__ long long operator()(int64_t i) const { return v[i] < cap ? v[i] : cap; }
};

__global__ void __launch_bounds__(256)
compact_hits_kernel(int64_t n_active, int max_hits, const int32_t *__restrict__ pixel_id,
                    const int32_t *__restrict__ slots, const int32_t *__restrict__ hits_per_pixel,
                    const int32_t *__restrict__ hit_off, long long *counters, int64_t hit_capacity,
                    int32_t *hit_pixel, int32_t *hit_tick, int32_t *hit_adc)
{
    const int64_t slot = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (slot >= n_active) return;
    const int cnt = hits_per_pixel[slot];
    const int m = cnt < max_hits ? cnt : max_hits;
    const int64_t base = counters[0] + hit_off[slot];
    int dropped = 0;
    for (int k = 0; k < m; ++k) {
        const int64_t h = base + k;
        if (h < hit_capacity) {
            const int v = slots[slot * max_hits + k];
            hit_pixel[h] = pixel_id[slot];
            hit_tick[h] = v >> ADC_SHIFT;
            hit_adc[h] = v & ((1 << ADC_SHIFT) - 1);
        } else ++dropped;
    }
    if (cnt > max_hits) atomicAdd((unsigned long long *)&counters[2], 1ull);
    if (cnt) atomicAdd((unsigned long long *)&counters[1], (unsigned long long)cnt);
    if (dropped) atomicAdd((unsigned long long *)&counters[3], (unsigned long long)dropped);
}

__global__ void advance_hit_base_kernel(long long *counters, const long long *batch_total, int64_t hit_capacity)
{
    long long v = counters[0] + *batch_total;
    counters[0] = v < hit_capacity ? v : hit_capacity;
}

// slot_scratch: int32[n_active * max_hits]; scan_scratch: int32[n_active] + one long long (aligned) after it
int launch_electronics(lartpc_sim *sim, const lartpc_waveforms_t *wf, uint64_t seed, lartpc_hits_t *out,
                       int32_t *slot_scratch, int32_t *scan_scratch, int64_t, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    const int64_t na = wf->n_active;
    if (na == 0) return LARTPC_OK;
    ++g_lartpc_launches;
    if (p.noise_disc != 0.0 || p.periodic > 0 || p.hold < 0)
        electronics_kernel<<<div_up(na, 128), 128, 0, st>>>(p, seed, na, wf->pixel_id, wf->first_tick, wf->length,
                                                           wf->offset, wf->samples, sim->disabled_mask, slot_scratch,
                                                           out->hits_per_pixel, out->q_pixel);
    else
        electronics_warp_kernel<<<div_up(na, 4), 128, 0, st>>>(p, seed, na, wf->pixel_id, wf->first_tick, wf->length,
                                                              wf->offset, wf->samples, sim->disabled_mask, slot_scratch,
                                                              out->hits_per_pixel, out->q_pixel);
    int rc = sim_ensure_scan_tmp(sim, na);
    if (rc) return rc;
    long long *batch_total = sim->d_counters + CNT_COUNT - 1;
    LARTPC_CUDA_TRY(lscan::exclusive_scan(na, HitCountF{out->hits_per_pixel, p.max_hits}, scan_scratch, false,
                                          batch_total, sim->scan_tmp, st));
    ++g_lartpc_launches;
    compact_hits_kernel<<<div_up(na, 256), 256, 0, st>>>(na, p.max_hits, wf->pixel_id, slot_scratch,
                                                        out->hits_per_pixel, scan_scratch, (long long *)out->counters,
                                                        out->hit_capacity, out->hit_pixel, out->hit_tick, out->hit_adc);
    ++g_lartpc_launches;
    advance_hit_base_kernel<<<1, 1, 0, st>>>((long long *)out->counters, batch_total, out->hit_capacity);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}


// -------------------------------------------------------------------------------------------------
// S6 without any allocation: lartpc_electronics_static (include/lartpc.h).  Same kernels and same launch order as
// launch_electronics above; what differs is where the scratch lives.  lartpc_electronics grows sim-owned buffers with
// cudaMalloc when a call needs more than the last one did (per-pixel hit slots, hit offsets, the prefix sum's block sums):
// a caller under CUDA graph capture, or one that must not allocate after start-up, cannot use that.  Here the scratch is
// one file-scope device array of a fixed, modest size that every GPU loading the library holds until the process ends;
// inputs beyond it are refused (LARTPC_ERR_STATIC_LIMIT), nothing is ever grown.
//   layout (bytes):  [0, 256)                    header: the batch's hit total (long long), written by the scan before it is read
//                    [256, 256 + 8 * 4096)       block sums of the prefix sum (long long; MAX_PIXELS / 2048 + 1 used)
//                    then int32 offs[MAX_PIXELS + 64], int32 slots[MAX_SLOTS]
// Every call (of every sim, every stream, every thread) shares the array: calls that overlap on the GPU race on it.  It
// keeps the last call's contents; every word a call reads it has written before (electronics kernel -> slots, scan ->
// block sums, offsets, total), the header is cleared all the same.
// In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address: the address the kernels
// get is resolved with cudaGetSymbolAddress, once per device, with that device current (static_scratch_ptr below: from
// lartpc_sim_create, and again -- a table look-up then -- by the entry point).
// -------------------------------------------------------------------------------------------------
constexpr int64_t STATIC_MAX_PIXELS = LARTPC_STATIC_MAX_PIXELS;
constexpr int64_t STATIC_MAX_SLOTS = LARTPC_STATIC_MAX_SLOTS;
constexpr size_t STATIC_HDR_BYTES = 256, STATIC_SUMS_BYTES = 8 * 4096;
constexpr size_t STATIC_OFFS_BYTES = sizeof(int32_t) * (size_t)(STATIC_MAX_PIXELS + 64);
constexpr size_t STATIC_SCRATCH_BYTES = STATIC_HDR_BYTES + STATIC_SUMS_BYTES + STATIC_OFFS_BYTES + sizeof(int32_t) * (size_t)STATIC_MAX_SLOTS;
static_assert(STATIC_MAX_PIXELS / lscan::TILE + 2 <= (int64_t)(STATIC_SUMS_BYTES / 8), "block sums of the largest accepted scan fit");
static_assert((STATIC_HDR_BYTES + STATIC_SUMS_BYTES + STATIC_OFFS_BYTES) % 256 == 0, "the slots start on a 256-byte boundary");

static __device__ __align__(256) unsigned char g_static_scratch[STATIC_SCRATCH_BYTES];

namespace {
constexpr int STATIC_MAX_DEVICES = 64;
void *g_static_ptr[STATIC_MAX_DEVICES];          // device address of g_static_scratch on device i (null: not resolved yet)
}

// device address of the scratch on `device`, which must be the current device; resolved once per device
int static_scratch_ptr(int device, void **ptr)
{
    if (device < 0 || device >= STATIC_MAX_DEVICES) return LARTPC_ERR_BAD_ARGUMENT;
    void *p = __atomic_load_n(&g_static_ptr[device], __ATOMIC_ACQUIRE);
    if (!p) {
        LARTPC_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_scratch));   // (idempotent: two threads racing here store the same address)
        if (!p) return LARTPC_ERR_CUDA;
        __atomic_store_n(&g_static_ptr[device], p, __ATOMIC_RELEASE);
    }
    *ptr = p;
    return LARTPC_OK;
}

extern "C" int lartpc_electronics_static(lartpc_sim_t *sim, const lartpc_waveforms_t *wf, uint64_t seed, lartpc_hits_t *out,
                                         void *stream)
{
    if (!sim || !wf || !out || !out->counters) return LARTPC_ERR_BAD_ARGUMENT;
    if (wf->n_active > 0 && (!out->hits_per_pixel || !out->q_pixel)) return LARTPC_ERR_BAD_ARGUMENT;
    const DevParams &p = sim->dp;
    const int64_t na = wf->n_active;
    if (na < 0) return LARTPC_ERR_BAD_ARGUMENT;
    if (na > STATIC_MAX_PIXELS || na * (int64_t)p.max_hits > STATIC_MAX_SLOTS) return LARTPC_ERR_STATIC_LIMIT;
    DeviceGuard dg(sim->device);
    cudaStream_t st = (cudaStream_t)stream;
    void *base = nullptr;
    int rc = static_scratch_ptr(sim->device, &base);
    if (rc) return rc;
    unsigned char *b = (unsigned char *)base;
    long long *batch_total = (long long *)b;
    long long *scan_tmp = (long long *)(b + STATIC_HDR_BYTES);
    int32_t *offs = (int32_t *)(b + STATIC_HDR_BYTES + STATIC_SUMS_BYTES);
    int32_t *slots = (int32_t *)(b + STATIC_HDR_BYTES + STATIC_SUMS_BYTES + STATIC_OFFS_BYTES);
    LARTPC_CUDA_TRY(cudaMemsetAsync(out->counters, 0, sizeof(int64_t) * 4, st));
    LARTPC_CUDA_TRY(cudaMemsetAsync(b, 0, STATIC_HDR_BYTES, st));
    if (na == 0) return LARTPC_OK;
    ++g_lartpc_launches;
    if (p.noise_disc != 0.0 || p.periodic > 0 || p.hold < 0)
        electronics_kernel<<<div_up(na, 128), 128, 0, st>>>(p, seed, na, wf->pixel_id, wf->first_tick, wf->length,
                                                           wf->offset, wf->samples, sim->disabled_mask, slots,
                                                           out->hits_per_pixel, out->q_pixel);
    else
        electronics_warp_kernel<<<div_up(na, 4), 128, 0, st>>>(p, seed, na, wf->pixel_id, wf->first_tick, wf->length,
                                                              wf->offset, wf->samples, sim->disabled_mask, slots,
                                                              out->hits_per_pixel, out->q_pixel);
    LARTPC_CUDA_TRY(lscan::exclusive_scan(na, HitCountF{out->hits_per_pixel, p.max_hits}, offs, false, batch_total, scan_tmp, st));
    ++g_lartpc_launches;
    compact_hits_kernel<<<div_up(na, 256), 256, 0, st>>>(na, p.max_hits, wf->pixel_id, slots, out->hits_per_pixel, offs,
                                                        (long long *)out->counters, out->hit_capacity, out->hit_pixel,
                                                        out->hit_tick, out->hit_adc);
    ++g_lartpc_launches;
    advance_hit_base_kernel<<<1, 1, 0, st>>>((long long *)out->counters, batch_total, out->hit_capacity);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}


// -------------------------------------------------------------------------------------------------
// Packed hit output (BASELINE configs[3] "16-bit packed hit output", reading D18): the (pixel, tick)-sorted hit list
// regrouped by readout tile (tile_pixels x tile_pixels pixels: 70 x 70) as three uint16 per hit
// {pixel in tile = iy_in * tile_pixels + ix_in, tick, adc | flags << 12}, with an offset table per tile.
// One CTA per readout tile; a pixel row of a tile is a contiguous run of the sorted list, found by binary search, so
// the order inside a tile is (pixel in tile, tick) and nothing depends on atomics.
// -------------------------------------------------------------------------------------------------
struct PackGeom { const DevTpc *tpcs; const int32_t *tile_base; int n_tpcs, tile_pixels; };

__device__ __forceinline__ int64_t lower_bound_i32(const int32_t *v, int64_t n, int32_t key)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) {
        const int64_t mid = (lo + hi) >> 1;
        if (v[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

template <bool WRITE>
__global__ void __launch_bounds__(128)
pack_hits_kernel(PackGeom g, int64_t n_hits, const int32_t *__restrict__ hit_pixel, const int32_t *__restrict__ hit_tick,
                 const int32_t *__restrict__ hit_adc, int32_t *tile_count, const int64_t *__restrict__ tile_off,
                 uint16_t *packed)
{
    __shared__ long long s_start[256];
    __shared__ int s_cnt[256], s_pre[257];
    const int tile = blockIdx.x, tid = threadIdx.x;
    int tpc = 0;
    while (tpc + 1 < g.n_tpcs && g.tile_base[tpc + 1] <= tile) ++tpc;
    const DevTpc &t = g.tpcs[tpc];
    const int tp = g.tile_pixels, ntx = (t.nx + tp - 1) / tp;
    const int rel = tile - g.tile_base[tpc], ty = rel / ntx, tx = rel - ty * ntx;
    const int x0 = tx * tp, x1 = min(x0 + tp, t.nx), y0 = ty * tp, rows = min(y0 + tp, t.ny) - y0;
    for (int r = tid; r < rows; r += blockDim.x) {
        const int32_t id0 = t.first_pixel_id + (y0 + r) * t.nx + x0, id1 = id0 + (x1 - x0);
        const int64_t a = lower_bound_i32(hit_pixel, n_hits, id0), b = lower_bound_i32(hit_pixel, n_hits, id1);
        s_start[r] = a;  s_cnt[r] = (int)(b - a);
    }
    __syncthreads();
    if (tid == 0) {
        int run = 0;
        for (int r = 0; r < rows; ++r) { s_pre[r] = run; run += s_cnt[r]; }
        s_pre[rows] = run;
        if (!WRITE) tile_count[tile] = run;
    }
    if (!WRITE) return;
    __syncthreads();
    const int64_t base = tile_off[tile];
    for (int r = 0; r < rows; ++r) {
        const int64_t src = s_start[r];
        for (int k = tid; k < s_cnt[r]; k += blockDim.x) {
            const int64_t h = src + k;
            const int32_t id = hit_pixel[h] - t.first_pixel_id;
            const int iy = id / t.nx, ix = id - iy * t.nx;
            uint16_t *o = packed + 3 * (base + s_pre[r] + k);
            o[0] = (uint16_t)((iy - y0) * tp + (ix - x0));
            o[1] = (uint16_t)hit_tick[h];
            o[2] = (uint16_t)(hit_adc[h] & 0x0fff);
        }
    }
}

struct TileCountF { const int32_t *v; __device__ long long operator()(int64_t i) const { return v[i]; } };

int launch_pack_hits(lartpc_sim *sim, const lartpc_hits_t *hits, int64_t n_hits, int tile_pixels, uint16_t *packed,
                     int64_t *tile_offsets, cudaStream_t st)
{
    const DevParams &p = sim->dp;
    // readout tiles per TPC, in table order
    std::vector<int32_t> base(p.n_tpcs + 1, 0);
    for (int k = 0; k < p.n_tpcs; ++k) {
        const lartpc_tpc_t &t = sim->tpcs[k];
        base[k + 1] = base[k] + ((t.nx + tile_pixels - 1) / tile_pixels) * ((t.ny + tile_pixels - 1) / tile_pixels);
    }
    const int n_rt = base[p.n_tpcs];
    if (sim->pack_tile_pixels != tile_pixels) {
        cudaFree(sim->pack_base);  cudaFree(sim->pack_count);
        sim->pack_base = nullptr;  sim->pack_count = nullptr;  sim->pack_tile_pixels = 0;
        LARTPC_CUDA_TRY(cudaMalloc(&sim->pack_base, sizeof(int32_t) * (p.n_tpcs + 1)));
        LARTPC_CUDA_TRY(cudaMalloc(&sim->pack_count, sizeof(int32_t) * (n_rt + 1)));
        LARTPC_CUDA_TRY(cudaMemcpy(sim->pack_base, base.data(), sizeof(int32_t) * (p.n_tpcs + 1), cudaMemcpyHostToDevice));
        sim->pack_tile_pixels = tile_pixels;
    }
    int rc = sim_ensure_scan_tmp(sim, n_rt);
    if (rc) return rc;
    PackGeom g{sim->d_tpcs, sim->pack_base, p.n_tpcs, tile_pixels};
    g_lartpc_launches += 2;
    pack_hits_kernel<false><<<n_rt, 128, 0, st>>>(g, n_hits, hits->hit_pixel, hits->hit_tick, hits->hit_adc,
                                                  sim->pack_count, nullptr, nullptr);
    LARTPC_CUDA_TRY(lscan::exclusive_scan((int64_t)n_rt, TileCountF{sim->pack_count}, tile_offsets, true,
                                          (long long *)nullptr, sim->scan_tmp, st));
    pack_hits_kernel<true><<<n_rt, 128, 0, st>>>(g, n_hits, hits->hit_pixel, hits->hit_tick, hits->hit_adc,
                                                 sim->pack_count, tile_offsets, packed);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}
