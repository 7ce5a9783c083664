/*
 * lartpc.h -- C-ABI boundary of the B200-native charge-readout hot path of the pixelated
 * LArTPC simulation of arXiv 2212.09807 (P:L### = line of /root/reference/PAPER.md).
 *
 * Path:  segments S_i = (r_s, r_e, E)_i  (eq. 2.1)
 *   S1 lartpc_quench               recombination, eqs. (3.1)/(3.2)
 *   S2 lartpc_drift                drift time, lifetime, diffusion, eqs. (3.3)-(3.5)
 *   S3 lartpc_pixels_from_segments pixel / tick pre-sizing
 *   S4 lartpc_induced_current      eq. (3.9) against the response LUT
 *   S5 lartpc_sum_pixel_signals    per-pixel sum over tracks
 *   S6 lartpc_electronics          LArPix CSA / discriminator / 8-bit ADC / noise
 *   S7 lartpc_run_spill            S1..S6 streamed in TPC batches
 *
 * Conventions
 *   - Plain C, no C++/torch types.  Every pointer inside a lartpc_*_t bundle is a DEVICE pointer
 *     allocated and owned by the caller unless the field comment says "host".  The library owns
 *     only what lartpc_sim_create copies (response LUT, TPC table) plus internal planning scratch
 *     sized by the geometry and grown on demand (tile lists); see lartpc_sim_t.
 *   - Units: cm, us, MeV, electrons, mV; ticks are integers of params.tick_us.
 *   - All stage calls enqueue work on `stream` (a cudaStream_t passed as void*; NULL = default
 *     stream).  S1, S2, S4, S6 return without synchronising.  S3 and S5 (plan mode) synchronise the
 *     stream once because they report data-dependent sizes to the host, as the paper's pre-sizing
 *     step does.  lartpc_run_spill synchronises internally per TPC batch.
 *   - Return value: 0 = LARTPC_OK, negative = error (lartpc_strerror).  Nothing is thrown or
 *     aborted across the ABI.  Capacity overflows found on the device (hit list full, more than
 *     max_hits_per_pixel hits on a pixel) are counted in the output bundle / stats and never write
 *     out of bounds.
 *   - There is no CPU fallback and no dispatch: lartpc_sim_create fails unless the current device
 *     has compute capability 10.x.  The library reads no environment variable: which kernel runs is decided by
 *     the parameters and the response mode alone.
 *   - A lartpc_sim_t holds the plan made by S3 for ONE batch of segments; S4/S5/S6 must follow on
 *     the same sim, in order, before the next S3.  A sim is not re-entrant across streams.
 */
#ifndef LARTPC_H
#define LARTPC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LARTPC_OK                 0
#define LARTPC_ERR_BAD_ARGUMENT  (-1)
#define LARTPC_ERR_CAPACITY      (-2)   /* a caller buffer is too small; the needed size is reported */
#define LARTPC_ERR_CUDA          (-3)
#define LARTPC_ERR_LUT_SHAPE     (-4)
#define LARTPC_ERR_DEVICE        (-5)   /* not a compute-capability 10.x device */
#define LARTPC_ERR_UNSUPPORTED   (-6)
#define LARTPC_ERR_ORDER         (-7)   /* stage called without the plan of the preceding stage */
#define LARTPC_ERR_STATIC_LIMIT  (-8)   /* input larger than the fixed scratch of lartpc_electronics_static */

typedef struct lartpc_sim lartpc_sim_t;   /* opaque: LUT copy, TPC table, planning scratch */

/* All physics constants as doubles so that both sides of a parity test start from identical values.
 * Defaults in brackets. */
typedef struct {
    double e_field_kv_cm, lar_density_g_cm3, w_ion_mev;        /* [0.5, 1.38, 23.6e-6] */
    int    recomb_model;                                       /* 0 = Birks eq. (3.1), 1 = modified Box eq. (3.2) */
    double birks_ab, birks_kb, box_alpha, box_beta;            /* [0.800, 0.0486, 0.93, 0.212 | 0.207] */
    double v_drift_cm_us, lifetime_us;                         /* [0.16, 2200] */
    double d_long_cm2_us, d_tran_cm2_us;                       /* [4.0e-6, 8.8e-6] = 4.0, 8.8 cm^2/s */
    double tick_us, t_origin_us;                               /* [0.1, 0]; arrival tick j = floor((T - t_origin)/tick) */
    double pixel_pitch_cm;                                     /* [0.4434] */
    int    bins_per_pixel, window_pixels, lut_ticks;           /* nb [10], W [5 | 9, odd], K [200..2000, multiple of 4] */
    int    n_readout_ticks;                                    /* readout ticks n = j + k, n in [0, n_readout_ticks) */
    double sample_step_cm, n_sigma_map;                        /* [1e-3 = 10 um, 5.0] */
    double gain_mv_per_ke, v_cm_mv, v_ref_mv, v_pedestal_mv;   /* [4, 288, 1300, 580] */
    int    adc_bits;                                           /* [8] */
    double threshold_e;                                        /* [7000] = 28 mV */
    int    hold_ticks, min_spacing_ticks, periodic_reset_ticks;/* [16, 11, 0 = off] */
    double noise_reset_e, noise_disc_e, noise_uncorr_e;        /* [0|900, 0|650, 0|500] */
    int    max_hits_per_pixel;                                 /* capacity of the per-pixel hit scratch [32] */
} lartpc_params_t;

/* One TPC drift volume and its pixel plane.  Plane-local u = x - x0, v = y - y0; drift along z:
 * d(z) = clamp(drift_sign * (z - z_anode), 0, drift_len) (eq. 3.3 with a sign for two-sided modules,
 * P:L830).  Pixel (ix, iy) has global id first_pixel_id + iy * nx + ix. */
typedef struct {
    double x0, y0, z_anode;
    int    drift_sign;          /* +1 or -1 */
    double drift_len;
    int    nx, ny;
    int    first_pixel_id;
} lartpc_tpc_t;

/* Input: structure-of-arrays segments, each array float32[n] (eq. 2.1). */
typedef struct {
    const float *xs, *ys, *zs, *ts;     /* start point (cm) and time (us) */
    const float *xe, *ye, *ze, *te;     /* end point and time */
    const float *dE;                    /* deposited energy (MeV) */
} lartpc_segments_t;

/* S2 output, each array [n].  Endpoints stay in float64 so that the diffusion weights of S4 do not
 * lose the sub-micron position of a segment on a 3 m plane ("fp32 cancellation"). */
typedef struct {
    int32_t *tpc;                       /* TPC index, -1 = midpoint in no TPC (inactive, D8) */
    float   *q_anode;                   /* Q_a = n_e exp(-t_mid/tau), electrons (eq. 3.4) */
    float   *sigma_T;                   /* transverse sigma, cm (eq. 3.5 with D_T) */
    float   *sigma_t;                   /* longitudinal sigma as a time, us (sigma_L / v_drift) */
    double  *u_s, *v_s, *u_e, *v_e;     /* plane-local endpoints, cm */
    double  *T_s, *T_e;                 /* anode arrival times of the two ends, us */
} lartpc_drifted_t;

/* S3 output, each array int32[n] except offsets int64[n+1].  All integers are bit-exact functions of
 * the float32 inputs (float64 IEEE arithmetic in a fixed order). */
typedef struct {
    int32_t *a_lo, *a_hi, *b_lo, *b_hi; /* charged-bin box (bin = pitch / bins_per_pixel), inclusive */
    int32_t *ix0, *ix1, *iy0, *iy1;     /* pixel rectangle, inclusive; empty when ix0 > ix1 */
    int32_t *jt0, *jt1;                 /* arrival-tick range, inclusive (not clipped to the window) */
    int32_t *npix;                      /* pixels in the rectangle */
    int32_t *n_samples;                 /* N = max(1, ceil(L / sample_step)) */
    int64_t *offsets;                   /* exclusive scan of npix, [n+1] */
} lartpc_pixmap_t;

/* S3 host-side report (the paper's "longest signal / largest number of pixels") plus the sizes
 * the caller needs to allocate the S4/S5/S6 outputs. */
typedef struct {
    int32_t max_npix;                   /* largest rectangle */
    int32_t max_ticks;                  /* longest signal: max(jt1 - jt0 + 1) + lut_ticks - 1 */
    int64_t total_npix;                 /* offsets[n] */
    int64_t n_active_segments;          /* segments with a non-empty rectangle */
    int64_t n_tiles;                    /* charge tiles (charged pixel x window of arrival ticks) S4 will process */
    int64_t n_pairs;                    /* (segment, charged pixel) incidences */
    int64_t n_active_pixels;            /* pixels that can receive current */
    int64_t total_samples;              /* sum of the per-pixel waveform lengths S5 will write */
    int32_t tile_targets;               /* W*W: partial waveforms per tile */
    int32_t tile_ticks;                 /* readout ticks per partial waveform (padded) */
    int32_t tile_charge_floats;         /* 32-bit words of one tile's packed charge lattice (lartpc_signals_t.charge) */
    int32_t tile_block;                 /* the charge buffer must hold n_tiles rounded up to a multiple of this (256 with the
                                           tensor-core response: two 128-tile MMA blocks per CTA pair; 1 otherwise) */
} lartpc_pixmap_info_t;

/* S4 output.  A tile is (charged pixel P, window of lartpc_chunk_ticks() arrival ticks that starts at
 * j_start = first arrival tick on P, rounded down to a multiple of 4, + a multiple of the window length).
 *   charge      the charge lattice of eq. (3.8) in expectation, C[bin][j] electrons per (x, y) LUT bin of P and
 *               arrival tick, tile_charge_floats 32-bit words per tile.
 *               Tensor-core response (lartpc_response_mode() == LARTPC_RESPONSE_TENSOR): the operand image the MMAs
 *               read, [slot / 128][bin][16-tick block][fp16 part | fp8 part][slot % 128][32 bytes], where a tile's
 *               slot is given by the sim's plan (tiles that charge the same 16-tick blocks sit together); the fp16
 *               part holds C 2^-e, the fp8 (e4m3) part {lo8 = (C 2^-e - fp16 part) 2^5, hi8 = C 2^-e 2^-7} per tick,
 *               e in tile_range; blocks no tile of a 256-slot unit (the two 128-tile blocks a CTA pair multiplies at once)
 *               charges are neither written nor read; the buffer must hold a whole number of units: tile_capacity >=
 *               n_tiles rounded up to lartpc_pixmap_info_t.tile_block.
 *               FFMA response: packed per tile as a header (bins, charge groups, first / last output block), one
 *               item per non-empty bin (bin, first tick, groups of 4 ticks, row offset) and the charge rows;
 *   partial     float32 [n_tiles][tile_targets][tile_ticks] (electrons per tick), indexed by slot: the current that
 *               charge induces on the W x W pixels around P during readout ticks [j_start, j_start + tile_ticks);
 *               tile_targets = W*W, except on the tensor-core path with lut_ticks > 209, where the LUT is cut into
 *               pieces of 200 ticks and row (target d, piece q) = d * pieces + q covers ticks from j_start + 200 q;
 *   tile_range  int32 [n_tiles][4], indexed by slot = first / last 14-tick block of `partial` that can be non-zero
 *               (first > last: no charge), the scale exponent e, 0.
 * The tile -> pixel and tile -> slot maps are part of the sim's plan (FFMA response: slot = tile). */
typedef struct {
    int64_t  tile_capacity;             /* host value: tiles the charge buffer can hold (partial / tile_range: n_tiles) */
    float   *partial;
    int32_t *tile_range;
    float   *charge;
} lartpc_signals_t;

/* S5 output: one waveform per active pixel, sorted by pixel id. */
typedef struct {
    int64_t  pixel_capacity;            /* host values: capacities of the arrays below */
    int64_t  sample_capacity;
    int32_t *pixel_id;                  /* [n_active] sorted unique global pixel ids */
    int32_t *first_tick;                /* [n_active] readout tick of samples[offset] */
    int32_t *length;                    /* [n_active] */
    int64_t *offset;                    /* [n_active + 1] */
    float   *samples;                   /* [total_samples] electrons per tick */
    int64_t  n_active;                  /* host value, set by lartpc_sum_pixel_signals */
    int64_t  total_samples;             /* host value, set by lartpc_sum_pixel_signals */
} lartpc_waveforms_t;

/* S6 output: compact hit list sorted by (pixel id, tick). */
typedef struct {
    int64_t  hit_capacity;              /* host value */
    int32_t *hit_pixel;                 /* [hit_capacity] global pixel id */
    int32_t *hit_tick;                  /* [hit_capacity] digitisation tick (D14) */
    int32_t *hit_adc;                   /* [hit_capacity] ADC count 0 .. 2^adc_bits - 1 */
    int32_t *hits_per_pixel;            /* [n_active] all hits, also those beyond max_hits_per_pixel */
    float   *q_pixel;                   /* [n_active] Q_p = sum_n I_p[n], electrons */
    int64_t *counters;                  /* device int64[4]: n_hits written, n_hits total, pixels over
                                           max_hits_per_pixel, hits dropped for hit_capacity */
} lartpc_hits_t;

/* Truth association (reading D26): per hit the k_max segments with the largest shares. */
typedef struct {
    int32_t  k_max;                     /* host value: entries per hit, 1 .. 64 */
    int32_t  reserved;
    int32_t *seg;                       /* [n_hits][k_max] segment index (into the arrays given to S2 / S3), -1 = unused entry */
    float   *frac;                      /* [n_hits][k_max] q_{h,s} / q_signal[h]; entries by decreasing |q_{h,s}|, ties by index */
    float   *q_signal;                  /* [n_hits] sum over ALL segments of q_{h,s}: the charge the sample holds, without noise */
    int32_t *n_contrib;                 /* [n_hits] segments with a non-zero share */
} lartpc_truth_t;

typedef struct {
    int64_t n_segments, n_active_segments, n_tiles, n_pairs, n_active_pixels, total_samples;
    int64_t n_hits, n_hits_total, n_pixels_overflow, n_hits_dropped;
    int32_t n_batches;
    int32_t reserved;
    double  flops_current;              /* FMA * 2 issued by the S4 response + splat loops (counted on the host
                                           from the plan; 0 when not computed) */
} lartpc_stats_t;

/* ---- lifetime -------------------------------------------------------------------------------- */

/* Copies params, the TPC table and the response LUT (HOST pointer, float32 [W*nb][W*nb][K], tick
 * fastest, R[cy][cx][k] = electrons induced during LUT tick k on the centre pixel of the W x W window by
 * one electron above bin (cx, cy) that arrives during LUT tick K-1, D4, D5).  lut_elems must
 * equal (W*nb)^2 * K (else LARTPC_ERR_LUT_SHAPE).  Values: any finite float32 in any units; the tensor-core response
 * scales the table by a power of two chosen from max |R| (so a table in other units than the harness's "electrons per
 * electron" keeps the same relative accuracy); a NaN or infinite entry is LARTPC_ERR_BAD_ARGUMENT.  Entries below
 * 2^-21 max |R| keep their value to fp16-subnormal precision only (absolute error <= 2^-35 max |R|).
 * The sim lives on the CUDA device that is current at creation; every later call runs there whatever the caller's
 * current device is (several sims on several devices may coexist in one process). */
int  lartpc_sim_create(const lartpc_params_t *params, const lartpc_tpc_t *tpcs, int n_tpcs,
                       const float *response_lut_host, size_t lut_elems, lartpc_sim_t **out);
void lartpc_sim_destroy(lartpc_sim_t *sim);

/* As lartpc_sim_create, choosing how S4 applies the response (eq. 3.7):
 *   LARTPC_RESPONSE_TENSOR  dense contraction of the charge lattice with the LUT on the tcgen05 tensor cores, operands
 *                           split hi + lo (fp16 main term, fp8 cross terms, fp32 accumulation); a LUT longer than
 *                           209 ticks is applied in pieces of 200 ticks; window_pixels^2 <= 128;
 *   LARTPC_RESPONSE_FFMA    sliding-window convolution on the FP32 pipe (packed FFMA2), any LUT shape;
 *   LARTPC_RESPONSE_AUTO    TENSOR where it applies, else FFMA (what lartpc_sim_create does).
 * Both give the same currents within the S4 tolerance; LARTPC_ERR_UNSUPPORTED when TENSOR
 * is asked for a LUT it cannot take. */
#define LARTPC_RESPONSE_AUTO   0
#define LARTPC_RESPONSE_TENSOR 1
#define LARTPC_RESPONSE_FFMA   2
int  lartpc_sim_create_ex(const lartpc_params_t *params, const lartpc_tpc_t *tpcs, int n_tpcs,
                          const float *response_lut_host, size_t lut_elems, int response_mode, lartpc_sim_t **out);
/* LARTPC_RESPONSE_TENSOR or LARTPC_RESPONSE_FFMA: the path this sim runs. */
int  lartpc_response_mode(const lartpc_sim_t *sim);

/* Optional mask of disabled channels: HOST array of global pixel ids; S6 emits no hit for them. */
int  lartpc_set_disabled_pixels(lartpc_sim_t *sim, const int32_t *pixel_ids_host, int64_t n);

/* Eq. (3.9) as printed: m > 0 makes S4 perturb each of the N sample points of a
 * segment m times, (dx, dy) ~ N(0, sigma_T), dt ~ N(0, sigma_t), and look the LUT up at the nearest bin and tick of every
 * perturbed point (charge Q_a / (N m) each), instead of taking the perturbation in expectation (m = 0, the default;
 * DESIGN.md reading D1).  The normals of point (segment index s, mu, nu) are Box-Muller pairs of Philox4x32-10 with
 * counter (s, mu, nu, 0x52414E44) and key (seed lo, seed hi), clamped to +- n_sigma_map (reading D25).  m <= 255.
 * Tensor-core path with 5 or 10 bins per pixel only: LARTPC_ERR_UNSUPPORTED otherwise. */
int  lartpc_set_random_perturbations(lartpc_sim_t *sim, int m, uint64_t seed);

/* Tensor-core response only.  tcgen05.mma adds every product into its fp32 accumulator with truncation toward zero
 * (measured on B200: the integrated current of a pixel comes out low by 0.4 - 1.4e-5 of its gross value, growing with the
 * number of charged LUT cells), a systematic loss that fp32 FMA accumulation (round to nearest) does not have and that
 * moves hits across ADC code boundaries where a pixel's gross current is large.  The response's epilogue multiplies
 * accumulator column n by 1 + kappa x (non-zero charge cells whose products that column summed), the expected loss;
 * kappa = LARTPC_TRUNC_KAPPA_DEFAULT, measured against the fp64 oracle on configs[1..3] (residual bias <= 1.5e-6, rms
 * <= 3.5e-6 of gross; reading D27), unless set here; 0 turns the compensation off.  0 <= kappa <= 1e-6. */
#define LARTPC_TRUNC_KAPPA_DEFAULT 7.5e-9
int  lartpc_set_truncation_compensation(lartpc_sim_t *sim, double kappa);

/* Arrival ticks per charge tile (window length) chosen for this LUT shape. */
int  lartpc_chunk_ticks(const lartpc_sim_t *sim);

/* Recommended workspace for lartpc_run_spill on up to max_segments segments. */
size_t lartpc_workspace_bytes(const lartpc_sim_t *sim, int64_t max_segments);

/* ---- stages ---------------------------------------------------------------------------------- */

/* S1 (eqs. 3.1/3.2): dEdx[n] MeV/cm, n_e[n] electrons after recombination. */
int  lartpc_quench(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n,
                   float *dEdx, float *n_e, void *stream);

/* S2 (eqs. 3.3-3.5). */
int  lartpc_drift(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n, const float *n_e,
                  lartpc_drifted_t *out, void *stream);

/* S3: pixel rectangles, tick ranges, sample counts; builds the sim's tile plan; fills *info (host)
 * after one stream synchronisation. */
int  lartpc_pixels_from_segments(lartpc_sim_t *sim, const lartpc_segments_t *seg,
                                 const lartpc_drifted_t *drifted, int64_t n,
                                 lartpc_pixmap_t *out, lartpc_pixmap_info_t *info, void *stream);

/* S4: needs out->tile_capacity >= info.n_tiles rounded up to info.tile_block.  Two kernels: the
 * charge lattice of every tile (splat), then the response of the W x W pixels around it (persistent; tensor cores, or
 * LUT rows streamed through shared memory for the FFMA form). */
int  lartpc_induced_current(lartpc_sim_t *sim, const lartpc_drifted_t *drifted, const lartpc_pixmap_t *pixmap,
                            int64_t n, lartpc_signals_t *out, void *stream);

/* S5: needs pixel_capacity >= info.n_active_pixels and sample_capacity >= info.total_samples. */
int  lartpc_sum_pixel_signals(lartpc_sim_t *sim, const lartpc_signals_t *signals,
                              lartpc_waveforms_t *out, void *stream);

/* S6: Philox4x32-10 noise keyed by (seed, pixel id, tick). */
int  lartpc_electronics(lartpc_sim_t *sim, const lartpc_waveforms_t *waveforms, uint64_t seed,
                        lartpc_hits_t *out, void *stream);

/* S6 for callers that must not allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * the same kernels, the same launch order and the same results as lartpc_electronics, bit for bit -- but where that call
 * grows sim-owned scratch with cudaMalloc whenever a call needs more than the last one did, this one keeps its scratch
 * (per-pixel hit slots, hit offsets, block sums of the prefix sum) in ONE file-scope device array of fixed size
 * (~8.3 MB, held by every GPU that loads the library until the process exits) and calls no cudaMalloc, cudaFree or
 * allocating library routine, ever.  Limits: waveforms->n_active <= LARTPC_STATIC_MAX_PIXELS and n_active x
 * max_hits_per_pixel <= LARTPC_STATIC_MAX_SLOTS (65 536 active pixels at the default 32 hits per pixel: configs[0], [1] and a
 * TPC of configs[2] / [3]); beyond them LARTPC_ERR_STATIC_LIMIT, nothing launched, nothing written.  Inputs and outputs are
 * the caller's, exactly as for lartpc_electronics.  The array is shared by every call of every sim, stream and thread of
 * the process on that GPU and keeps the last call's contents (each call writes what it reads before reading it): calls
 * that OVERLAP on the GPU race on it -- order them on one stream, or with events. */
#define LARTPC_STATIC_MAX_PIXELS 65536
#define LARTPC_STATIC_MAX_SLOTS  2097152
int  lartpc_electronics_static(lartpc_sim_t *sim, const lartpc_waveforms_t *waveforms, uint64_t seed,
                               lartpc_hits_t *out, void *stream);

/* Truth association, an optional pass after S6 (the paper has it for the light path; reading D26).  By
 * eqs. (3.7)-(3.9) the current on a pixel is a sum over segments; the share of segment s in hit h of pixel p is
 *     q_{h,s} = sum_{n = n0}^{n_h} I_{p,s}[n],   I_{p,s} = eq. (3.9) for segment s alone,
 * over the ticks the CSA integrated for that sample: n_h = hit_tick, n0 = hit_tick of the pixel's previous hit + 1 (0 for
 * its first), or a later periodic-reset tick <= n_h - hold_ticks.  Shares are signed (bipolar induced currents); noise
 * belongs to no segment.  `hits` must be sorted by (pixel, tick) as S6 / S7 write it, n_hits its length; drifted / pixmap /
 * n are those the sim's current plan (S3) was made from (LARTPC_ERR_ORDER otherwise: after lartpc_run_spill the plan holds
 * the last TPC batch only, so use the staged calls).  Not available with lartpc_set_random_perturbations (m > 0).
 * Accuracy: a share is within max(1e-4 |q|, 1 e-) of the fp64 value (same weights as S4).  Cost: one pass over the charge
 * cells of every (hit, segment, source pixel): seconds at configs[3] scale, it is not part of lartpc_run_spill. */
int  lartpc_hit_truth(lartpc_sim_t *sim, const lartpc_drifted_t *drifted, const lartpc_pixmap_t *pixmap, int64_t n,
                      const lartpc_hits_t *hits, int64_t n_hits, lartpc_truth_t *out, void *stream);

/* S7: the whole path on device-resident segments; hits of all batches are appended to *out in
 * (pixel id, tick) order per batch (batches are TPC ranges, so the list is globally sorted).
 * out->hits_per_pixel and out->q_pixel may be NULL. */
int  lartpc_run_spill(lartpc_sim_t *sim, const lartpc_segments_t *seg, int64_t n, uint64_t seed,
                      lartpc_hits_t *out, lartpc_stats_t *stats, void *workspace, size_t ws_bytes,
                      void *stream);

/* Packed hit output (BASELINE configs[3]: "16-bit packed hit output"; reading D18).  Regroups a hit list
 * sorted by (pixel id, tick) -- what lartpc_electronics / lartpc_run_spill write -- by readout tile of tile_pixels x
 * tile_pixels pixels (70 in the paper; <= 255), tiles numbered TPC by TPC in table order, row-major inside a TPC
 * (planes whose size is not a multiple of tile_pixels end in partial tiles).  packed: device uint16[n_hits][3] =
 * {pixel in tile = iy_in * tile_pixels + ix_in, tick, adc | flags << 12 (flags = 0)}, ordered by (tile, pixel in tile,
 * tick); tile_offsets: device int64[lartpc_readout_tiles() + 1], hits of tile k are [tile_offsets[k], tile_offsets[k+1]).
 * Bit-exact, order-defined.  n_readout_ticks <= 65536 and adc_bits <= 12, else LARTPC_ERR_UNSUPPORTED. */
int64_t lartpc_readout_tiles(const lartpc_sim_t *sim, int tile_pixels);
int  lartpc_pack_hits(lartpc_sim_t *sim, const lartpc_hits_t *hits, int64_t n_hits, int tile_pixels,
                      uint16_t *packed, int64_t *tile_offsets, void *stream);

/* ---- light simulation (eqs. 4.1-4.6; readings D28-D33) ------------------
 * A second workload on the same segments: photons -> photoelectrons per photosensor -> time profile -> scintillation time
 * structure -> counting statistics -> read-out waveform.  The light look-up table (made with Geant4 in the paper)
 * is an input: visibility V_i[voxel] and relative arrival-time distribution f_i[voxel][time bin] per photosensor i over a
 * regular voxel grid.  All waveforms are float32 [n_det][n_ticks], tick fastest; every array argument is a DEVICE pointer
 * unless it says host.  The light trigger (serial by construction) and the final resampling are not part of it. */
typedef struct lartpc_light lartpc_light_t;   /* opaque: device copies of the tables, sorting scratch */

typedef struct {
    double w_ph_mev, w_ion_mev;             /* energy per photon at zero field [19.5e-6], per electron [23.6e-6] */
    double tick_us, t_start_us;             /* simulation tick delta_t [0.016] and the time of tick 0 */
    int    n_ticks;                         /* ticks of every waveform */
    int    lut_m, n_lut_t;                  /* a LUT time bin spans lut_m ticks (D29); LUT time bins */
    double vox_x0, vox_y0, vox_z0, vox_size_cm;   /* voxel grid: origin (cm) and voxel edge */
    int    nvx, nvy, nvz, n_det;            /* voxels per axis (x fastest), photosensors */
    double f_prompt, tau_prompt_us, tau_slow_us;  /* eq. (4.4): [0.3, 0.007, 1.6] */
    double trunc_tau;                       /* eq. (4.5) is truncated at trunc_tau * tau_slow [5] */
    double normal_above;                    /* Poisson below, normal at or above this many expected p.e. [30] */
    int    n_resp, n_noise;                 /* taps of the impulse response (sampled at the tick, D32); noise sinusoids (0: none) */
} lartpc_light_params_t;

/* Copies the tables (HOST pointers): eff[n_det] (eps_i of eq. 4.2), gain[n_det] (G_i of eq. 4.6), vis[n_det][nvz][nvy][nvx],
 * tprof[n_det][nvz][nvy][nvx][n_lut_t] (each profile sums to 1), resp[n_resp] (unit-normalised), noise_amp[n_noise] and
 * noise_k[n_noise] (amplitude and cycles per waveform of each noise sinusoid, D33; may be NULL when n_noise = 0).
 * LARTPC_ERR_BAD_ARGUMENT for non-positive sizes or ticks, LARTPC_ERR_DEVICE off compute capability 10.x. */
int  lartpc_light_create(const lartpc_light_params_t *params, const float *eff_host, const float *gain_host,
                         const float *vis_host, const float *tprof_host, const float *resp_host,
                         const float *noise_amp_host, const int32_t *noise_k_host, lartpc_light_t **out);
void lartpc_light_destroy(lartpc_light_t *light);

/* L1, eqs. (4.1)(4.2): N_gamma,j = dE_j / W_ph - n_e,j (n_e from lartpc_quench: the same recombination as the charge,
 * P:L736; clamped at 0), N_pe,ij = eps_i V_i[voxel of the midpoint of segment j] N_gamma,j (D28).  Out: vox[n] (voxel index,
 * -1 outside the grid: no light), k0[n] (tick of the deposition time (ts + te) / 2), n_gamma[n], npe[n_det][n]. */
int  lartpc_light_npe(lartpc_light_t *light, const lartpc_segments_t *seg, int64_t n, const float *n_e,
                      int32_t *vox, int32_t *k0, float *n_gamma, float *npe, void *stream);

/* L2, eq. (4.3) as read in D29: ipe[i][t] = photoelectrons reaching sensor i during tick t = sum over segments of
 * N_pe,ij f_i[vox_j][(t - k0_j) / lut_m] / lut_m.  Segments are sorted by deposition tick first (library scratch), every
 * (sensor, tick) then adds its contributions in a fixed order: bit-reproducible. */
int  lartpc_light_profile(lartpc_light_t *light, int64_t n, const int32_t *vox, const int32_t *k0, const float *npe,
                          float *ipe, void *stream);

/* L3, eqs. (4.4)(4.5): isc[i][t] = sum_{s=0}^{s_max} ipe[i][t-s] w[s], w[s] = integral of f_scint over tick s (D30),
 * s_max = floor(trunc_tau tau_slow / tick). */
int  lartpc_light_scintillation(lartpc_light_t *light, const float *ipe, float *isc, void *stream);

/* L4: nobs[i][t] = inverse-transform Poisson sample of isc[i][t] below normal_above, isc + sqrt(isc) z at or above;
 * uniforms from Philox4x32-10(counter (i, t, 0, 'LGHT'), key = seed) (D31); decisions in float64. */
int  lartpc_light_fluctuate(lartpc_light_t *light, uint64_t seed, const float *isc, float *nobs, void *stream);

/* L5, eq. (4.6): v[i][t] = n_i[t] + G_i sum_{s=0}^{n_resp-1} nobs[i][t-s] resp[s]; noise n_i as in D33 (keyed by seed). */
int  lartpc_light_electronics(lartpc_light_t *light, uint64_t seed, const float *nobs, float *v, void *stream);

/* L1..L5 on device-resident segments; intermediates live in `workspace` (lartpc_light_workspace_bytes(light, n) bytes,
 * LARTPC_ERR_CAPACITY if smaller).  v: float32 [n_det][n_ticks]. */
size_t lartpc_light_workspace_bytes(const lartpc_light_t *light, int64_t n);
int  lartpc_light_run(lartpc_light_t *light, const lartpc_segments_t *seg, int64_t n, const float *n_e, uint64_t seed,
                      float *v, void *workspace, size_t ws_bytes, void *stream);

/* ---- measurement aids ------------------------------------------------------------------------ */

/* Runs an FFMA-chain microbenchmark on `stream` and returns the measured FP32 rate in TFLOP/s
 * (2 flop per FMA) through *tflops; variant 0 = scalar FFMA, 1 = packed FFMA2.  Used as the
 * roofline denominator of S4. */
int  lartpc_measure_fp32_peak(int variant, double *tflops, void *stream);

/* Per-stage device times of lartpc_run_spill.  With profiling on, run_spill brackets every stage launch with
 * CUDA events recorded on `stream` and adds the elapsed times up per stage after its final synchronisation
 * (a few microseconds of overhead per launch; off by default).  lartpc_get_stage_ms returns, for the last
 * run_spill, ms[s] = device milliseconds and launches[s] = times the stage ran (one per TPC batch for S3-S6):
 * s = 0 quench, 1 drift, 2 pixel mapping + plan, 3 induced current: charge lattice, 4 induced current: response,
 * 5 per-pixel sum, 6 electronics.
 * fma_current = multiply-adds the S4 response needs for the charge it found (counted on the device:
 * non-zero charge cells x in-plane target pixels x lut_ticks), the numerator of its roofline figure. */
#define LARTPC_N_STAGES 7
int  lartpc_set_profiling(lartpc_sim_t *sim, int on);
int  lartpc_get_stage_ms(const lartpc_sim_t *sim, double ms[LARTPC_N_STAGES], int64_t launches[LARTPC_N_STAGES],
                         double *fma_current);

/* Work counters of the last lartpc_run_spill, counted on the device by the S4 kernels (the numerators of bench.py's
 * per-kernel roofline figures; tensor-core path):
 *   [0] multiply-adds the method needs: non-zero charge cells x in-plane target pixels x lut_ticks (= fma_current above)
 *   [1] tcgen05.mma instructions the response issued (each 128 tiles x NBW columns x 16 fp16 or 32 fp8 products deep)
 *   [2] bytes the response copied from L2 / HBM into shared memory (charge blocks + LUT generators)
 *   [3] operand columns (sample points / rule nodes x tiles) the charge lattice evaluated
 *   [4] tcgen05.mma instructions the charge lattice issued (128 cells x 64 ticks x 16 columns deep)
 *   [5] response work items (unit of tiles x target row) that held charge
 *   [6], [7] reserved (0) */
#define LARTPC_N_COUNTERS 8
int  lartpc_get_counters(const lartpc_sim_t *sim, double out[LARTPC_N_COUNTERS]);

/* Kernels the library has launched in this process so far (all sims; not thread-safe, a plain counter). */
int64_t lartpc_kernel_launches(void);

const char *lartpc_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* LARTPC_H */
