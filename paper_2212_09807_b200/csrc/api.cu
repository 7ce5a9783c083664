// C-ABI entry points of liblartpc (include/lartpc.h): sim lifetime, stage wrappers, the spill driver
// and the FP32 peak microbenchmark used as the roofline denominator of S4.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#include <algorithm>
#include <cmath>
#include <new>
#include "common.cuh"

size_t lartpc_splat_smem(const DevParams &p);
size_t lartpc_response_smem(const DevParams &p);

static thread_local char g_last_cuda_error[256] = "";
long long g_lartpc_launches = 0;

extern "C" int64_t lartpc_kernel_launches(void) { return (int64_t)g_lartpc_launches; }

void lartpc_note_cuda_error(cudaError_t e, const char *file, int line)
{
    snprintf(g_last_cuda_error, sizeof(g_last_cuda_error), "%s (%s:%d)", cudaGetErrorString(e), file, line);
    cudaGetLastError();
}

extern "C" const char *lartpc_strerror(int code)
{
    switch (code) {
        case LARTPC_OK: return "ok";
        case LARTPC_ERR_BAD_ARGUMENT: return "bad argument";
        case LARTPC_ERR_CAPACITY: return "caller buffer too small";
        case LARTPC_ERR_CUDA: return g_last_cuda_error[0] ? g_last_cuda_error : "CUDA error";
        case LARTPC_ERR_LUT_SHAPE: return "response LUT shape does not match (W*nb)^2 * K";
        case LARTPC_ERR_DEVICE: return "device is not compute capability 10.x (sm_100a only, no fallback)";
        case LARTPC_ERR_UNSUPPORTED: return "unsupported parameter combination";
        case LARTPC_ERR_ORDER: return "stage called out of order (no plan from lartpc_pixels_from_segments)";
        case LARTPC_ERR_STATIC_LIMIT:
            return "input exceeds the fixed scratch of lartpc_electronics_static (LARTPC_STATIC_MAX_PIXELS active pixels, "
                   "LARTPC_STATIC_MAX_SLOTS = n_active x max_hits_per_pixel hit slots); use lartpc_electronics";
        default: return "unknown error";
    }
}

static void sim_free(lartpc_sim *s)
{
    if (!s) return;
    DeviceGuard dg(s->device);
    cudaFree(s->d_tpcs); cudaFree(s->d_lut); cudaFree(s->d_lut_tc); cudaFree(s->d_cum_lut);
    cudaFree(s->pix_count); cudaFree(s->pix_start); cudaFree(s->pix_tile0); cudaFree(s->pix_cursor);
    cudaFree(s->pix_mask); cudaFree(s->act_first); cudaFree(s->act_last); cudaFree(s->act_slot);
    cudaFree(s->pair_seg); cudaFree(s->tile_cp); cudaFree(s->tile_desc); cudaFree(s->tile_list); cudaFree(s->cell_list); cudaFree(s->seg_rec);
    cudaFree(s->pack_base); cudaFree(s->pack_count);
    cudaFree(s->tile_perm); cudaFree(s->tile_desc_p); cudaFree(s->tile_list_p); cudaFree(s->tb_mask); cudaFree(s->tc_cmask); cudaFree(s->cls_hist); cudaFree(s->scan_tmp);
    cudaFree(s->d_counters); cudaFree(s->disabled_mask); cudaFree(s->elec_slots); cudaFree(s->elec_offs);
    cudaFree(s->d_fma); cudaFree(s->d_work); cudaFree(s->pix_jmin); cudaFree(s->d_end_row);
    for (cudaEvent_t e : s->ev_pool) cudaEventDestroy(e);
    if (s->h_counters) cudaFreeHost(s->h_counters);
    delete s;
}

extern "C" void lartpc_sim_destroy(lartpc_sim_t *sim) { sim_free(sim); }


// Output blocks at both ends of a tile have fewer taps inside [0, K) than the interior ones, and consumer threads are
// laid out slot-major (slot = tid / PG), so giving slot k block k would load the four SM sub-partitions (warp % 4)
// unevenly and the busiest one would set the pace.  Pick, once per geometry, the block of every slot by a seeded
// hill-climb that minimises the mean of max/mean sub-partition load over typical charge rows (1..16 groups).
static void balance_blocks(const DevParams &p, unsigned char *blk_of_slot)
{
    const int nblk = p.nblk_max, PG = p.PG, K = p.K;
    std::vector<int> perm(nblk);
    for (int b = 0; b < nblk; ++b) perm[b] = b;
    std::vector<double> share(4 * nblk, 0.0);
    for (int t = 0; t < PG * nblk && t < RESP_CONSUMERS; ++t) share[((t / 32) % 4) * nblk + t / PG] += 1.0;
    std::vector<std::vector<double>> prof;
    const int jb0s[4] = {0, 2, 6, 10};
    for (int ng = 1; ng <= 16; ++ng)
        for (int jb0 : jb0s) {
            std::vector<double> w(nblk);
            for (int b = 0; b < nblk; ++b) {
                const int n0 = RESP_NO * b;
                const int lo = std::max(0, (n0 - jb0 - K - 2 + 3) >> 2), hi = std::min(ng - 1, (n0 - jb0 + RESP_NO - 1) >> 2);
                w[b] = std::max(0, hi - lo + 1);
            }
            prof.push_back(w);
        }
    auto cost = [&](const std::vector<int> &pm) {
        double tot = 0.0;
        for (const auto &w : prof) {
            double mx = 0.0, sum = 0.0;
            for (int sp = 0; sp < 4; ++sp) {
                double l = 0.0;
                for (int k = 0; k < nblk; ++k) l += share[sp * nblk + k] * w[pm[k]];
                mx = std::max(mx, l);  sum += l;
            }
            if (sum > 0.0) tot += mx / (sum / 4.0);
        }
        return tot;
    };
    double best = cost(perm);
    uint64_t rng = 0x9E3779B97F4A7C15ull;
    auto next = [&]() { rng = rng * 6364136223846793005ull + 1442695040888963407ull; return (uint32_t)(rng >> 33); };
    for (int it = 0; it < 4000 && nblk > 1; ++it) {
        const int i = next() % nblk, j = next() % nblk;
        if (i == j) continue;
        std::swap(perm[i], perm[j]);
        const double c = cost(perm);
        if (c < best) best = c; else std::swap(perm[i], perm[j]);
    }
    for (int k = 0; k < 256; ++k) blk_of_slot[k] = (unsigned char)(k < nblk ? perm[k] : 255);
}

extern "C" int lartpc_sim_create(const lartpc_params_t *prm, const lartpc_tpc_t *tpcs, int n_tpcs,
                                 const float *lut_host, size_t lut_elems, lartpc_sim_t **out)
{
    return lartpc_sim_create_ex(prm, tpcs, n_tpcs, lut_host, lut_elems, LARTPC_RESPONSE_AUTO, out);
}

extern "C" int lartpc_sim_create_ex(const lartpc_params_t *prm, const lartpc_tpc_t *tpcs, int n_tpcs,
                                    const float *lut_host, size_t lut_elems, int response_mode, lartpc_sim_t **out)
{
    if (!prm || !tpcs || n_tpcs <= 0 || !lut_host || !out) return LARTPC_ERR_BAD_ARGUMENT;
    if (response_mode != LARTPC_RESPONSE_AUTO && response_mode != LARTPC_RESPONSE_TENSOR &&
        response_mode != LARTPC_RESPONSE_FFMA)
        return LARTPC_ERR_BAD_ARGUMENT;
    *out = nullptr;
    int dev = 0;
    cudaDeviceProp prop;
    LARTPC_CUDA_TRY(cudaGetDevice(&dev));
    LARTPC_CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major != 10) return LARTPC_ERR_DEVICE;
    const int nb = prm->bins_per_pixel, W = prm->window_pixels, K = prm->lut_ticks;
    if (nb < 1 || nb > 15 || W < 1 || (W & 1) == 0 || K < 1 || prm->n_readout_ticks < K || prm->tick_us <= 0 ||
        prm->pixel_pitch_cm <= 0 || prm->sample_step_cm <= 0 || prm->adc_bits < 1 || prm->adc_bits > 12 ||
        prm->max_hits_per_pixel < 1 || prm->hold_ticks < 0 || prm->v_drift_cm_us <= 0)
        return LARTPC_ERR_BAD_ARGUMENT;
    if (lut_elems != (size_t)W * nb * W * nb * K) return LARTPC_ERR_LUT_SHAPE;
    if (prm->n_readout_ticks >= (1 << 19)) return LARTPC_ERR_UNSUPPORTED;

    lartpc_sim *s = new (std::nothrow) lartpc_sim();
    if (!s) return LARTPC_ERR_BAD_ARGUMENT;
    s->params = *prm;
    s->tpcs.assign(tpcs, tpcs + n_tpcs);
    s->sm_count = prop.multiProcessorCount;
    s->device = dev;
    {
        // set-up of lartpc_electronics_static: the device address of its scratch on this (the current) device, resolved once
        // per device; a failure here is reported by that entry point, which tries again
        void *scratch = nullptr;
        (void)static_scratch_ptr(dev, &scratch);
    }
    DevParams &p = s->dp;
    memset(&p, 0, sizeof(p));
    p.eps = prm->e_field_kv_cm * prm->lar_density_g_cm3;  p.w_ion = prm->w_ion_mev;
    p.birks_ab = prm->birks_ab; p.birks_kb = prm->birks_kb; p.box_alpha = prm->box_alpha; p.box_beta = prm->box_beta;
    p.v_drift = prm->v_drift_cm_us; p.lifetime = prm->lifetime_us; p.d_long = prm->d_long_cm2_us;
    p.d_tran = prm->d_tran_cm2_us; p.dt = prm->tick_us; p.t_origin = prm->t_origin_us; p.pitch = prm->pixel_pitch_cm;
    p.bin = prm->pixel_pitch_cm / (double)nb;  p.sample_step = prm->sample_step_cm;  p.n_sigma_map = prm->n_sigma_map;
    p.recomb_model = prm->recomb_model;
    p.nb = nb; p.W = W; p.H = (W - 1) / 2; p.K = K; p.WW = W * W; p.NB2 = nb * nb;
    p.n_ticks = prm->n_readout_ticks;  p.j_max = p.n_ticks - K;
    // S4 geometry.  A response task is (pair of target pixels, RESP_NO output ticks); the consumer threads of one CTA
    // cover PG pairs x nblk_max blocks, and a tile needs n_groups passes to cover all pairs.  Jc (arrival ticks per
    // tile, multiple of 4, at most 120) is chosen to maximise the arrival ticks covered per pass.
    p.RS = LUT_OFF + K + 22;
    while ((p.RS & 1) != 0 || ((p.RS >> 1) & 1) == 0) ++p.RS;               // RS = 2 * odd: conflict-free LDS.128 rows
    const int n_pairs = (p.WW + 1) / 2, ncons = RESP_CONSUMERS;
    const size_t smem_limit = (size_t)prop.sharedMemPerBlockOptin;
    const int jc_cap = 120;
    double best = 0.0;
    int best_groups = 0;
    for (int g = 1; g <= n_pairs; ++g) {
        DevParams q = p;
        q.n_groups = g;  q.PG = (n_pairs + g - 1) / g;
        int jc = std::min(jc_cap, RESP_NO * (ncons / q.PG) - K + 1) & ~3;
        if (jc < 8) continue;
        q.Jc = jc;  q.CJ = jc + 4;
        q.nblk_max = (jc + K - 2) / RESP_NO + 1;
        if (q.nblk_max > 255) continue;
        if (lartpc_splat_smem(q) > smem_limit || lartpc_response_smem(q) > smem_limit) continue;
        const double score = (double)jc / g;
        if (score > best) { best = score; best_groups = g; }
    }
    // Tensor-core response (response_tc.cuh): tiles of 64 arrival ticks; even and odd 16-tick blocks have an accumulator
    // each (32 + NBW columns, NBW = roundup16(KQ + 15)), and the two must fit the 512 TMEM columns: NBW <= 224.  A LUT
    // longer than 209 ticks is cut into pieces of KQ = 200 ticks: piece q is a LUT of its own whose response lands
    // 200 q ticks later, one more row per (tile, target) in `partial`, which S5 adds like the rows of other tiles.
    const int kq = ((K + 15 + 15) & ~15) <= 224 ? K : 200, nq = (K + kq - 1) / kq;
    const int nbw = (kq + 15 + 15) & ~15;
    const bool tc_ok = p.WW <= 128 && (long long)p.WW * nq <= 4096;
    if (response_mode == LARTPC_RESPONSE_TENSOR && !tc_ok) { sim_free(s); return LARTPC_ERR_UNSUPPORTED; }
    p.tc_mode = (response_mode != LARTPC_RESPONSE_FFMA && tc_ok) ? 1 : 0;
    if (best_groups == 0 && !p.tc_mode) { sim_free(s); return LARTPC_ERR_UNSUPPORTED; }
    s->lut_copy.assign(lut_host, lut_host + lut_elems);
    if (p.tc_mode) {
        // operand scale of the LUT: a power of two that puts max |R| into (2^9, 2^10], whatever units the table is in
        // (fp16 operand, e4m3 cross-term parts: response_tc.cuh); a table with a non-finite entry is refused
        float mx = 0.f;
        for (size_t i = 0; i < lut_elems; ++i) {
            if (!std::isfinite(lut_host[i])) { sim_free(s); return LARTPC_ERR_BAD_ARGUMENT; }
            mx = std::max(mx, fabsf(lut_host[i]));
        }
        int e2 = 0;
        if (mx > 0.f) { frexpf(mx, &e2); if (ldexpf(1.f, e2 - 1) == mx) --e2; }   // mx in (2^(e2-1), 2^e2]
        p.b_scale_log2 = 10 - std::min(std::max(e2, -30), 30);
        p.NBW = nbw;  p.KQ = kq;  p.nq = nq;
        p.trunc_kappa = LARTPC_TRUNC_KAPPA_DEFAULT;
        p.n_groups = 1;  p.PG = n_pairs;  p.NP = n_pairs;                 // (unused by the tensor-core response)
        p.Jc = 64;  p.CJ = p.Jc + 4;
        p.tile_ticks = (p.Jc + kq - 1 + 7) & ~7;                          // 264 for K = 200: ticks of one row of `partial`
        p.nblk_max = (p.tile_ticks + RESP_NO - 1) / RESP_NO;
        p.slab_floats = p.NB2 * p.Jc;                                     // NB2 rows of (64 hi + 64 lo) fp16
        if (lartpc_splat_smem(p) > smem_limit) { sim_free(s); return LARTPC_ERR_UNSUPPORTED; }
    } else {
        p.n_groups = best_groups;  p.PG = (n_pairs + p.n_groups - 1) / p.n_groups;  p.NP = p.n_groups * p.PG;
        p.Jc = std::min(jc_cap, RESP_NO * (ncons / p.PG) - K + 1) & ~3;  p.CJ = p.Jc + 4;
        p.nblk_max = (p.Jc + K - 2) / RESP_NO + 1;  p.tile_ticks = RESP_NO * p.nblk_max;  p.KQ = K;  p.nq = 1;
        p.slab_floats = (((SLAB_HDR + 2 * p.NB2 + 3) & ~3) + p.NB2 * (4 + p.CJ) + 3) & ~3;
    }
    if (p.j_max / p.Jc + 2 > MAX_WINDOWS) {                                 // window masks are 128 bits
        sim_free(s);
        return LARTPC_ERR_UNSUPPORTED;
    }
    if (!p.tc_mode) balance_blocks(p, s->blk_of_slot);
    p.n_tpcs = n_tpcs;
    p.gain_mv_per_ke = prm->gain_mv_per_ke; p.v_cm = prm->v_cm_mv; p.v_ref = prm->v_ref_mv; p.v_ped = prm->v_pedestal_mv;
    p.adc_full = ldexp(1.0, prm->adc_bits);  p.threshold = prm->threshold_e;
    p.noise_reset = prm->noise_reset_e; p.noise_disc = prm->noise_disc_e; p.noise_uncorr = prm->noise_uncorr_e;
    p.hold = prm->hold_ticks; p.min_spacing = prm->min_spacing_ticks; p.periodic = prm->periodic_reset_ticks;
    p.max_hits = prm->max_hits_per_pixel;

    std::vector<DevTpc> dt(n_tpcs);
    int64_t cp = 0, pix = 0;
    s->cp_base_h.assign(n_tpcs + 1, 0);  s->pix_base_h.assign(n_tpcs + 1, 0);
    for (int k = 0; k < n_tpcs; ++k) {
        s->cp_base_h[k] = cp;  s->pix_base_h[k] = pix;
        const lartpc_tpc_t &t = tpcs[k];
        if (t.nx < 1 || t.ny < 1 || (t.drift_sign != 1 && t.drift_sign != -1) || t.drift_len < 0 ||
            t.first_pixel_id != pix) {                                      // pixel ids must be dense, in table order
            sim_free(s);
            return LARTPC_ERR_BAD_ARGUMENT;
        }
        DevTpc &d = dt[k];
        d.x0 = t.x0; d.y0 = t.y0; d.z_anode = t.z_anode; d.drift_len = t.drift_len;
        d.x1 = t.x0 + (double)t.nx * prm->pixel_pitch_cm;  d.y1 = t.y0 + (double)t.ny * prm->pixel_pitch_cm;
        d.sign = t.drift_sign; d.nx = t.nx; d.ny = t.ny; d.first_pixel_id = t.first_pixel_id;
        d.gw = t.nx + 2 * p.H; d.gh = t.ny + 2 * p.H; d.cp_base = (int)cp; d.pad = 0;
        cp += (int64_t)d.gw * d.gh;
        pix += (int64_t)t.nx * t.ny;
    }
    if (cp >= INT32_MAX || pix >= INT32_MAX) { sim_free(s); return LARTPC_ERR_UNSUPPORTED; }
    s->n_cp = cp; s->n_pix = pix;
    s->cp_base_h[n_tpcs] = cp;  s->pix_base_h[n_tpcs] = pix;

    // LUT re-laid out as [bin c = cb*nb+ca][pair q][RS][2]: pair q interleaves the rows of targets d = 2q and 2q+1
    // (d = dyi*W + dxi; row (c, d) is R[cy = nb*dyi + cb][cx = nb*dxi + ca][.]), LUT tick k at pair-word LUT_OFF + k
    // with zero padding around it.  S4 stages the PG pair rows of one bin with a single bulk copy, reads 20-tap windows
    // with aligned 128-bit loads and feeds both targets of a pair to one packed f32x2 multiply-add.
    std::vector<float> re(p.tc_mode ? 0 : (size_t)p.NB2 * p.NP * p.RS * 2, 0.f);
    const int NB = W * nb;
    for (int cb = 0; cb < nb && !p.tc_mode; ++cb)
        for (int ca = 0; ca < nb; ++ca)
            for (int dyi = 0; dyi < W; ++dyi)
                for (int dxi = 0; dxi < W; ++dxi) {
                    const int d = dyi * W + dxi;
                    const float *src = lut_host + ((size_t)(nb * dyi + cb) * NB + (nb * dxi + ca)) * K;
                    float *dst = re.data() + (((size_t)(cb * nb + ca) * p.NP + d / 2) * p.RS + LUT_OFF) * 2 + (d & 1);
                    for (int k = 0; k < K; ++k) dst[2 * k] = src[k];
                }
#define SIM_TRY(expr) do { cudaError_t _e = (expr); if (_e != cudaSuccess) { \
        lartpc_note_cuda_error(_e, __FILE__, __LINE__); sim_free(s); return LARTPC_ERR_CUDA; } } while (0)
    if (p.tc_mode) {
        if (lartpc_build_lut_tc(p, lut_host, &s->d_lut_tc) == 0) { sim_free(s); return LARTPC_ERR_CUDA; }
    } else {
        SIM_TRY(cudaMalloc(&s->d_lut, sizeof(float) * re.size()));
        SIM_TRY(cudaMemcpy(s->d_lut, re.data(), sizeof(float) * re.size(), cudaMemcpyHostToDevice));
    }
    SIM_TRY(cudaMalloc(&s->d_tpcs, sizeof(DevTpc) * n_tpcs));
    SIM_TRY(cudaMemcpy(s->d_tpcs, dt.data(), sizeof(DevTpc) * n_tpcs, cudaMemcpyHostToDevice));
    SIM_TRY(cudaMalloc(&s->pix_count, sizeof(int32_t) * cp));
    SIM_TRY(cudaMalloc(&s->pix_start, sizeof(int32_t) * cp));
    SIM_TRY(cudaMalloc(&s->pix_tile0, sizeof(int32_t) * cp));
    SIM_TRY(cudaMalloc(&s->pix_cursor, sizeof(int32_t) * cp));
    SIM_TRY(cudaMalloc(&s->pix_mask, sizeof(unsigned long long) * MASK_WORDS * cp));
    SIM_TRY(cudaMalloc(&s->pix_jmin, sizeof(int32_t) * cp));
    SIM_TRY(cudaMalloc(&s->d_work, sizeof(int)));
    {
        const int end_row[4] = {0, 0, 2, 0};                                // {first tick, groups, flags = END, tile}
        SIM_TRY(cudaMalloc(&s->d_end_row, sizeof(end_row)));
        SIM_TRY(cudaMemcpy(s->d_end_row, end_row, sizeof(end_row), cudaMemcpyHostToDevice));
    }
    SIM_TRY(cudaMalloc(&s->act_first, sizeof(int32_t) * pix));
    SIM_TRY(cudaMalloc(&s->act_last, sizeof(int32_t) * pix));
    SIM_TRY(cudaMalloc(&s->act_slot, sizeof(int32_t) * pix));
    SIM_TRY(cudaMalloc(&s->d_counters, sizeof(long long) * CNT_COUNT));
    SIM_TRY(cudaMallocHost(&s->h_counters, sizeof(long long) * CNT_COUNT));
    SIM_TRY(cudaMalloc(&s->d_fma, sizeof(unsigned long long) * LARTPC_N_COUNTERS));
    SIM_TRY(cudaMemset(s->d_fma, 0, sizeof(unsigned long long) * LARTPC_N_COUNTERS));
    s->pair_cap = 1 << 16;
    SIM_TRY(cudaMalloc(&s->pair_seg, sizeof(int32_t) * s->pair_cap));
    if (sim_grow_tiles(s, 1 << 14) != 0) { sim_free(s); return LARTPC_ERR_CUDA; }
#undef SIM_TRY
    *out = s;
    return LARTPC_OK;
}

extern "C" int lartpc_set_disabled_pixels(lartpc_sim_t *sim, const int32_t *ids, int64_t n)
{
    if (!sim || (n > 0 && !ids)) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    const size_t words = (size_t)(sim->n_pix + 31) / 32;
    std::vector<uint32_t> m(words, 0u);
    for (int64_t i = 0; i < n; ++i) {
        if (ids[i] < 0 || ids[i] >= sim->n_pix) return LARTPC_ERR_BAD_ARGUMENT;
        m[ids[i] >> 5] |= 1u << (ids[i] & 31);
    }
    if (!sim->disabled_mask) LARTPC_CUDA_TRY(cudaMalloc(&sim->disabled_mask, sizeof(uint32_t) * words));
    LARTPC_CUDA_TRY(cudaMemcpy(sim->disabled_mask, m.data(), sizeof(uint32_t) * words, cudaMemcpyHostToDevice));
    return LARTPC_OK;
}

extern "C" int lartpc_set_random_perturbations(lartpc_sim_t *sim, int m, uint64_t seed)
{
    if (!sim || m < 0 || m > 255) return LARTPC_ERR_BAD_ARGUMENT;
    // the one-hot columns of the perturbed points exist in the tensor-core charge lattice only
    if (m > 0 && !splat_on_tc(sim->dp)) return LARTPC_ERR_UNSUPPORTED;
    sim->dp.rnd_m = m;
    sim->dp.rnd_seed = seed;
    sim->have_signals = false;
    return LARTPC_OK;
}

extern "C" int lartpc_set_truncation_compensation(lartpc_sim_t *sim, double kappa)
{
    if (!sim || !(kappa >= 0.0) || kappa > 1e-6) return LARTPC_ERR_BAD_ARGUMENT;
    sim->dp.trunc_kappa = (float)kappa;
    return LARTPC_OK;
}

extern "C" int64_t lartpc_readout_tiles(const lartpc_sim_t *sim, int tile_pixels)
{
    if (!sim || tile_pixels < 1 || tile_pixels > 255) return LARTPC_ERR_BAD_ARGUMENT;
    int64_t n = 0;
    for (const lartpc_tpc_t &t : sim->tpcs)
        n += (int64_t)((t.nx + tile_pixels - 1) / tile_pixels) * ((t.ny + tile_pixels - 1) / tile_pixels);
    return n;
}

extern "C" int lartpc_pack_hits(lartpc_sim_t *sim, const lartpc_hits_t *hits, int64_t n_hits, int tile_pixels,
                                uint16_t *packed, int64_t *tile_offsets, void *stream)
{
    if (!sim || !hits || n_hits < 0 || tile_pixels < 1 || tile_pixels > 255 || !tile_offsets || (n_hits > 0 && !packed))
        return LARTPC_ERR_BAD_ARGUMENT;
    if (n_hits > 0 && (!hits->hit_pixel || !hits->hit_tick || !hits->hit_adc)) return LARTPC_ERR_BAD_ARGUMENT;
    if (sim->dp.n_ticks > 65536 || sim->params.adc_bits > 12) return LARTPC_ERR_UNSUPPORTED;   // tick and adc must fit 16 / 12 bits
    DeviceGuard dg(sim->device);
    return launch_pack_hits(sim, hits, n_hits, tile_pixels, packed, tile_offsets, (cudaStream_t)stream);
}

extern "C" int lartpc_chunk_ticks(const lartpc_sim_t *sim) { return sim ? sim->dp.Jc : 0; }
extern "C" int lartpc_response_mode(const lartpc_sim_t *sim)
{
    return sim ? (sim->dp.tc_mode ? LARTPC_RESPONSE_TENSOR : LARTPC_RESPONSE_FFMA) : LARTPC_ERR_BAD_ARGUMENT;
}

// ---- stage wrappers -------------------------------------------------------------------------------
extern "C" int lartpc_quench(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n, float *dEdx, float *n_e,
                             void *stream)
{
    if (!sim || !seg || n < 0 || (n > 0 && (!dEdx || !n_e))) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    return launch_quench(sim, seg, n, dEdx, n_e, (cudaStream_t)stream);
}

extern "C" int lartpc_drift(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n, const float *n_e,
                            lartpc_drifted_t *out, void *stream)
{
    if (!sim || !seg || n < 0 || !out || (n > 0 && !n_e)) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    return launch_drift(sim, seg, n, n_e, out, (cudaStream_t)stream);
}

extern "C" int lartpc_pixels_from_segments(lartpc_sim_t *sim, const lartpc_segments_t *seg,
                                           const lartpc_drifted_t *dr, int64_t n, lartpc_pixmap_t *out,
                                           lartpc_pixmap_info_t *info, void *stream)
{
    if (!sim || !seg || !dr || !out || n < 0) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    return launch_plan(sim, seg, dr, n, 0, sim->dp.n_tpcs, out, info, (cudaStream_t)stream);
}

extern "C" int lartpc_induced_current(lartpc_sim_t *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm,
                                      int64_t n, lartpc_signals_t *out, void *stream)
{
    if (!sim || !dr || !pm || !out) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    if (!sim->have_plan || n != sim->plan_n) return LARTPC_ERR_ORDER;
    if (out->tile_capacity < tiles_alloc(sim->dp, sim->n_tiles)) return LARTPC_ERR_CAPACITY;
    if (sim->n_tiles > 0 && (!out->partial || !out->tile_range || !out->charge)) return LARTPC_ERR_BAD_ARGUMENT;
    int rc = launch_current_splat(sim, dr, pm, n, out, (cudaStream_t)stream);
    if (rc == 0) rc = sim->dp.tc_mode ? launch_current_response_tc(sim, out, (cudaStream_t)stream)
                                       : launch_current_response(sim, out, (cudaStream_t)stream);
    if (rc == 0) sim->have_signals = true;
    return rc;
}

extern "C" int lartpc_hit_truth(lartpc_sim_t *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n,
                                const lartpc_hits_t *hits, int64_t n_hits, lartpc_truth_t *out, void *stream)
{
    if (!sim || !dr || !pm || !hits || !out || n_hits < 0 || out->k_max < 1 || out->k_max > 64) return LARTPC_ERR_BAD_ARGUMENT;
    if (n_hits > 0 && (!hits->hit_pixel || !hits->hit_tick || !out->seg || !out->frac || !out->q_signal || !out->n_contrib))
        return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    if (!sim->have_plan || n != sim->plan_n) return LARTPC_ERR_ORDER;
    return launch_hit_truth(sim, dr, pm, hits, n_hits, out, (cudaStream_t)stream);
}

extern "C" int lartpc_sum_pixel_signals(lartpc_sim_t *sim, const lartpc_signals_t *sig, lartpc_waveforms_t *out,
                                        void *stream)
{
    if (!sim || !sig || !out) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    if (!sim->have_plan || !sim->have_signals) return LARTPC_ERR_ORDER;
    if (out->pixel_capacity < sim->n_active || out->sample_capacity < sim->total_samples) return LARTPC_ERR_CAPACITY;
    return launch_sum(sim, sig, out, (cudaStream_t)stream);
}

static int ensure_i32(int32_t **p, int64_t *cap, int64_t need)
{
    if (need <= *cap) return LARTPC_OK;
    if (*p) cudaFree(*p);
    *p = nullptr;
    LARTPC_CUDA_TRY(cudaMalloc(p, sizeof(int32_t) * (need + need / 4 + 256)));
    *cap = need + need / 4 + 256;
    return LARTPC_OK;
}

extern "C" int lartpc_electronics(lartpc_sim_t *sim, const lartpc_waveforms_t *wf, uint64_t seed, lartpc_hits_t *out,
                                  void *stream)
{
    if (!sim || !wf || !out || !out->counters) return LARTPC_ERR_BAD_ARGUMENT;
    if (wf->n_active > 0 && (!out->hits_per_pixel || !out->q_pixel)) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    cudaStream_t st = (cudaStream_t)stream;
    LARTPC_CUDA_TRY(cudaMemsetAsync(out->counters, 0, sizeof(int64_t) * 4, st));
    // the per-pixel hit slots live in sim-owned scratch, grown on demand (no allocation after warm-up)
    int rc;
    if ((rc = ensure_i32(&sim->elec_slots, &sim->elec_slots_cap, wf->n_active * sim->dp.max_hits)) != 0) return rc;
    if ((rc = ensure_i32(&sim->elec_offs, &sim->elec_offs_cap, wf->n_active + 1)) != 0) return rc;
    return launch_electronics(sim, wf, seed, out, sim->elec_slots, sim->elec_offs, 0, st);
}

// ---- S7 spill driver ------------------------------------------------------------------------------
namespace {
struct Arena {
    char *base; size_t size, used;
    template <typename T> T *take(int64_t n)
    {
        size_t bytes = ((size_t)(n > 0 ? n : 1) * sizeof(T) + 255) & ~(size_t)255;
        if (used + bytes > size) return nullptr;
        T *p = (T *)(base + used);
        used += bytes;
        return p;
    }
};
}  // namespace

// stage timing: event pairs recorded around each stage launch when profiling is on
struct StageTimer {
    lartpc_sim *sim; cudaStream_t st; size_t used = 0;
    cudaEvent_t next()
    {
        if (used == sim->ev_pool.size()) {
            cudaEvent_t e;
            cudaEventCreate(&e);
            sim->ev_pool.push_back(e);
        }
        return sim->ev_pool[used++];
    }
    void begin(int stage)
    {
        if (!sim->profiling) return;
        sim->ev_stage.push_back(stage);
        cudaEventRecord(next(), st);
    }
    void end()
    {
        if (sim->profiling) cudaEventRecord(next(), st);
    }
    void collect()                        // after the stream has been synchronised
    {
        for (int s = 0; s < LARTPC_N_STAGES; ++s) { sim->stage_ms[s] = 0.0; sim->stage_launches[s] = 0; }
        for (size_t i = 0; i < sim->ev_stage.size(); ++i) {
            float ms = 0.f;
            cudaEventElapsedTime(&ms, sim->ev_pool[2 * i], sim->ev_pool[2 * i + 1]);
            sim->stage_ms[sim->ev_stage[i]] += ms;
            sim->stage_launches[sim->ev_stage[i]] += 1;
        }
        sim->ev_stage.clear();
    }
};

extern "C" int lartpc_set_profiling(lartpc_sim_t *sim, int on)
{
    if (!sim) return LARTPC_ERR_BAD_ARGUMENT;
    sim->profiling = on != 0;
    return LARTPC_OK;
}

extern "C" int lartpc_get_stage_ms(const lartpc_sim_t *sim, double ms[LARTPC_N_STAGES],
                                   int64_t launches[LARTPC_N_STAGES], double *fma_current)
{
    if (!sim || !ms) return LARTPC_ERR_BAD_ARGUMENT;
    for (int s = 0; s < LARTPC_N_STAGES; ++s) {
        ms[s] = sim->stage_ms[s];
        if (launches) launches[s] = sim->stage_launches[s];
    }
    if (fma_current) *fma_current = sim->fma_current;
    return LARTPC_OK;
}

extern "C" int lartpc_get_counters(const lartpc_sim_t *sim, double out[LARTPC_N_COUNTERS])
{
    if (!sim || !out) return LARTPC_ERR_BAD_ARGUMENT;
    for (int k = 0; k < LARTPC_N_COUNTERS; ++k) out[k] = sim->counters[k];
    return LARTPC_OK;
}

extern "C" size_t lartpc_workspace_bytes(const lartpc_sim_t *sim, int64_t max_segments)
{
    if (!sim) return 0;
    // per segment: n_e, dEdx (8) + drifted (64) + pixmap (12*4 + 8) = 128 B, rounded up to 160.  The tile buffers
    // (packed charge + partial waveforms, ~58 KB per tile for 5x5 x 200) and the waveforms of the largest TPC batch
    // depend on the data; on the BASELINE configs there are up to ~1.5 tiles per segment of a batch, so 2 GiB +
    // 16 KiB per segment lets run_spill take several TPCs per batch; it halves its batches until they fit whatever
    // it is given (one TPC of configs[3] needs ~6 GiB).
    // (a LUT cut into pieces has one partial row per piece: 26.4 KB more per tile and piece)
    return (size_t)max_segments * (160 + 16384 + (size_t)(sim->dp.tc_mode ? sim->dp.nq - 1 : 0) * 40000) + ((size_t)2 << 30);
}

extern "C" int lartpc_run_spill(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n, uint64_t seed,
                                lartpc_hits_t *out, lartpc_stats_t *stats, void *workspace, size_t ws_bytes,
                                void *stream)
{
    if (!sim || !seg || !out || !out->counters || !workspace || n < 0) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(sim->device);
    cudaStream_t st = (cudaStream_t)stream;
    const DevParams &p = sim->dp;
    Arena ar{(char *)workspace, ws_bytes, 0};
    lartpc_stats_t stt;
    memset(&stt, 0, sizeof(stt));
    stt.n_segments = n;
    LARTPC_CUDA_TRY(cudaMemsetAsync(out->counters, 0, sizeof(int64_t) * 4, st));
    LARTPC_CUDA_TRY(cudaMemsetAsync(sim->d_fma, 0, sizeof(unsigned long long) * LARTPC_N_COUNTERS, st));
    StageTimer tm{sim, st};
    sim->ev_stage.clear();

    float *dEdx = ar.take<float>(n), *n_e = ar.take<float>(n);
    lartpc_drifted_t dr;
    dr.tpc = ar.take<int32_t>(n); dr.q_anode = ar.take<float>(n); dr.sigma_T = ar.take<float>(n);
    dr.sigma_t = ar.take<float>(n);
    dr.u_s = ar.take<double>(n); dr.v_s = ar.take<double>(n); dr.u_e = ar.take<double>(n); dr.v_e = ar.take<double>(n);
    dr.T_s = ar.take<double>(n); dr.T_e = ar.take<double>(n);
    lartpc_pixmap_t pm;
    pm.a_lo = ar.take<int32_t>(n); pm.a_hi = ar.take<int32_t>(n); pm.b_lo = ar.take<int32_t>(n);
    pm.b_hi = ar.take<int32_t>(n); pm.ix0 = ar.take<int32_t>(n); pm.ix1 = ar.take<int32_t>(n);
    pm.iy0 = ar.take<int32_t>(n); pm.iy1 = ar.take<int32_t>(n); pm.jt0 = ar.take<int32_t>(n);
    pm.jt1 = ar.take<int32_t>(n); pm.npix = ar.take<int32_t>(n); pm.n_samples = ar.take<int32_t>(n);
    pm.offsets = ar.take<int64_t>(n + 1);
    if (!pm.offsets || !dEdx) return LARTPC_ERR_CAPACITY;
    const size_t mark = ar.used;

    int rc;
    tm.begin(0);
    if ((rc = launch_quench(sim, seg, n, dEdx, n_e, st)) != 0) return rc;
    tm.end();
    tm.begin(1);
    if ((rc = launch_drift(sim, seg, n, n_e, &dr, st)) != 0) return rc;
    tm.end();

    // batches of consecutive TPCs; a batch whose tiles / waveforms do not fit the workspace is halved
    int tpc_lo = 0;
    // batch size that fitted this workspace last time (a sizing hint like the plan buffers' capacities: a wrong hint only
    // costs a halving or leaves memory unused, never changes a result)
    int batch = (sim->batch_hint > 0 && sim->batch_hint_ws == ws_bytes) ? std::min(sim->batch_hint, p.n_tpcs) : p.n_tpcs;
    while (tpc_lo < p.n_tpcs) {
        int tpc_hi = std::min(p.n_tpcs, tpc_lo + batch);
        lartpc_pixmap_info_t info;
        tm.begin(2);
        if ((rc = launch_plan(sim, seg, &dr, n, tpc_lo, tpc_hi, &pm, &info, st)) != 0) return rc;
        tm.end();
        ar.used = mark;
        lartpc_signals_t sig;
        sig.tile_capacity = tiles_alloc(p, info.n_tiles);
        sig.partial = ar.take<float>(info.n_tiles * p.WW * p.nq * p.tile_ticks);
        sig.tile_range = ar.take<int32_t>(info.n_tiles * TILE_META);
        sig.charge = ar.take<float>(sig.tile_capacity * p.slab_floats);
        lartpc_waveforms_t wf;
        wf.pixel_capacity = info.n_active_pixels;  wf.sample_capacity = info.total_samples;
        wf.pixel_id = ar.take<int32_t>(info.n_active_pixels);
        wf.first_tick = ar.take<int32_t>(info.n_active_pixels);
        wf.length = ar.take<int32_t>(info.n_active_pixels);
        wf.offset = ar.take<int64_t>(info.n_active_pixels + 1);
        wf.samples = ar.take<float>(info.total_samples);
        int32_t *slots = ar.take<int32_t>(info.n_active_pixels * p.max_hits);
        int32_t *offs = ar.take<int32_t>(info.n_active_pixels + 2);
        lartpc_hits_t h = *out;
        h.hits_per_pixel = ar.take<int32_t>(info.n_active_pixels);
        h.q_pixel = ar.take<float>(info.n_active_pixels);
        if (!sig.partial || !sig.tile_range || !sig.charge || !wf.samples || !slots || !offs || !h.q_pixel) {
            if (tpc_hi - tpc_lo <= 1) return LARTPC_ERR_CAPACITY;       // one TPC does not fit the workspace
            batch = std::max(1, (tpc_hi - tpc_lo) / 2);
            continue;
        }
        if (tpc_lo == 0) { stt.n_active_segments = info.n_active_segments;  sim->batch_hint = batch;  sim->batch_hint_ws = ws_bytes; }
        stt.n_tiles += info.n_tiles;  stt.n_pairs += info.n_pairs;
        stt.n_active_pixels += info.n_active_pixels;  stt.total_samples += info.total_samples;
        stt.n_batches += 1;
        tm.begin(3);
        if ((rc = launch_current_splat(sim, &dr, &pm, n, &sig, st)) != 0) return rc;
        tm.end();
        tm.begin(4);
        if ((rc = p.tc_mode ? launch_current_response_tc(sim, &sig, st) : launch_current_response(sim, &sig, st)) != 0)
            return rc;
        tm.end();
        sim->have_signals = true;
        tm.begin(5);
        if ((rc = launch_sum(sim, &sig, &wf, st)) != 0) return rc;
        tm.end();
        tm.begin(6);
        if ((rc = launch_electronics(sim, &wf, seed, &h, slots, offs, 0, st)) != 0) return rc;
        tm.end();
        tpc_lo = tpc_hi;
    }
    long long hc[4];
    unsigned long long cnt[LARTPC_N_COUNTERS] = {};
    LARTPC_CUDA_TRY(cudaMemcpyAsync(hc, out->counters, sizeof(hc), cudaMemcpyDeviceToHost, st));
    LARTPC_CUDA_TRY(cudaMemcpyAsync(cnt, sim->d_fma, sizeof(cnt), cudaMemcpyDeviceToHost, st));
    LARTPC_CUDA_TRY(cudaStreamSynchronize(st));
    tm.collect();
    for (int k = 0; k < LARTPC_N_COUNTERS; ++k) sim->counters[k] = (double)cnt[k];
    sim->fma_current = (double)cnt[0];
    stt.flops_current = 2.0 * (double)cnt[0];
    stt.n_hits = hc[0]; stt.n_hits_total = hc[1]; stt.n_pixels_overflow = hc[2]; stt.n_hits_dropped = hc[3];
    if (stats) *stats = stt;
    return LARTPC_OK;
}

// ---- FP32 peak microbenchmark (roofline denominator of S4) -----------------------------
template <int VARIANT>
__global__ void __launch_bounds__(256) fp32_peak_kernel(float *sink, int iters, float seed)
{
    if (VARIANT == 0) {
        float a[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = seed + (float)(threadIdx.x + i);
        const float b = 0.999f, c = 1e-3f;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], b, c);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += a[i];
        if (s == 123.456f) sink[0] = s;
    } else {
        float2 a[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = make_float2(seed + (float)(threadIdx.x + i), seed - (float)i);
        const float2 b = make_float2(0.999f, 0.998f), c = make_float2(1e-3f, 2e-3f);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int r = 0; r < 8; ++r)
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    unsigned long long av, bv, cv;
                    av = *(unsigned long long *)&a[i]; bv = *(const unsigned long long *)&b; cv = *(const unsigned long long *)&c;
                    asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(av) : "l"(av), "l"(bv), "l"(cv));
                    a[i] = *(float2 *)&av;
                }
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 8; ++i) s += a[i].x + a[i].y;
        if (s == 123.456f) sink[0] = s;
    }
}

extern "C" int lartpc_measure_fp32_peak(int variant, double *tflops, void *stream)
{
    if (!tflops || variant < 0 || variant > 1) return LARTPC_ERR_BAD_ARGUMENT;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    LARTPC_CUDA_TRY(cudaGetDevice(&dev));
    LARTPC_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    float *sink = nullptr;
    LARTPC_CUDA_TRY(cudaMalloc(&sink, 16));
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int iters = 4096, blocks = sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        if (variant == 0) { ++g_lartpc_launches; fp32_peak_kernel<0><<<blocks, threads, 0, st>>>(sink, iters, 1.0f); }
        else { ++g_lartpc_launches; fp32_peak_kernel<1><<<blocks, threads, 0, st>>>(sink, iters, 1.0f); }
        cudaEventRecord(e1, st);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double fma = (double)blocks * threads * iters * 128.0;       // 8 rounds x 16 FMA per thread per iteration
        double tf = 2.0 * fma / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink);
    LARTPC_CUDA_TRY(cudaGetLastError());
    *tflops = best;
    return LARTPC_OK;
}
