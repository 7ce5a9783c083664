// Internal definitions shared by the sm_100a kernels of liblartpc (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/lartpc.h"

#define LARTPC_CUDA_TRY(expr)                                   \
    do {                                                        \
        cudaError_t _e = (expr);                                \
        if (_e != cudaSuccess) { lartpc_note_cuda_error(_e, __FILE__, __LINE__); return LARTPC_ERR_CUDA; } \
    } while (0)

void lartpc_note_cuda_error(cudaError_t e, const char *file, int line);
extern long long g_lartpc_launches;   // kernels launched by the library in this process (lartpc_kernel_launches)

// ---- constants copied to every kernel by value ------------------------------------------------
struct DevParams {
    // recombination / transport (float64: the index path must be IEEE-exact)
    double eps, w_ion, birks_ab, birks_kb, box_alpha, box_beta;
    double v_drift, lifetime, d_long, d_tran, dt, t_origin, pitch, bin, sample_step, n_sigma_map;
    int recomb_model;
    int nb, W, H, K, WW, NB2;        // bins per pixel, window pixels, half window, LUT ticks, W*W, nb*nb
    int n_ticks, j_max;              // readout ticks, last arrival tick inside the window (n_ticks - K)
    int Jc, CJ;                      // arrival ticks per charge tile; row stride of the tile's charge lattice (Jc + 4)
    int nblk_max, tile_ticks;        // output blocks of RESP_NO ticks per tile, RESP_NO * nblk_max
    int RS;                          // padded LUT row length in pair-words: [20 zeros][K][>= 22 zeros], RS = 2 * odd
    int PG, NP;                      // target pairs per consumer group; pairs incl. padding = n_groups * PG
    int n_groups;                    // pair groups per tile = response passes over a tile (1 for W = 5, K = 200)
    int slab_floats;                 // packed charge lattice of one tile: header, bin items, charge rows
                                     // (tensor-core mode: NB2 * 64 = the tile's rows of the fp16 hi / lo operand image)
    int rnd_m;                       // > 0: eq. (3.9) as printed, M random perturbations per sample point (lartpc_set_random_perturbations)
    unsigned long long rnd_seed;
    int tc_mode;                     // 1: S4 response on the tensor cores (response_tc.cuh), 0: packed-FFMA2 response
    int NBW;                         // tensor-core mode: output columns per 16-tick arrival block, roundup16(KQ + 15)
    int b_scale_log2;                // tensor-core mode: the LUT operand is R * 2^b_scale_log2, chosen per LUT so that max |R| lands
                                     // in (2^9, 2^10] (fp16 / e4m3 range of the fixed part splits, response_tc.cuh)
    float trunc_kappa;               // tensor-core mode: expected relative loss per accumulated product to the truncating fp32
                                     // accumulation of tcgen05.mma, added back by the response's epilogue (0 = off)
    int KQ, nq;                      // tensor-core mode: LUT ticks per piece and pieces (K <= 209: one piece of K ticks; longer
                                     // LUTs are cut into pieces of 200 ticks, each a row of its own in `partial`, added by S5)
    int n_tpcs;
    // electronics
    double gain_mv_per_ke, v_cm, v_ref, v_ped, adc_full, threshold;
    double noise_reset, noise_disc, noise_uncorr;
    int hold, min_spacing, periodic, max_hits;
};

struct DevTpc {
    double x0, y0, x1, y1, z_anode, drift_len;
    int sign, nx, ny, first_pixel_id;
    int gw, gh;                      // charged-pixel grid (nx + 2H) x (ny + 2H): charge just outside the
    int cp_base;                     // plane still acts on in-plane pixels
    int pad;
};

// TPC that holds global pixel id gp / charged-pixel cell cp: the table is sorted by both (binary search: a full-size
// detector has 70 TPCs, and the linear walk every thread of S5 did at its start was 13 % of that kernel)
__device__ __forceinline__ int tpc_of_pixel(const DevTpc *__restrict__ tpcs, int n_tpcs, long long gp)
{
    int lo = 0, hi = n_tpcs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((long long)tpcs[mid].first_pixel_id <= gp) lo = mid; else hi = mid - 1;
    }
    return lo;
}
__device__ __forceinline__ int tpc_of_cell(const DevTpc *__restrict__ tpcs, int n_tpcs, long long cp)
{
    int lo = 0, hi = n_tpcs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if ((long long)tpcs[mid].cp_base <= cp) lo = mid; else hi = mid - 1;
    }
    return lo;
}

struct SegPtrs { const float *xs, *ys, *zs, *ts, *xe, *ye, *ze, *te, *dE; };

// charge tile = (charged pixel, window of Jc arrival ticks starting at j_start = first tick of the pixel + win * Jc)
struct TileDesc { int tpc, px, py, j_start; };

constexpr int MASK_WORDS = 2;        // window masks are 128 bits per charged pixel
constexpr int MAX_WINDOWS = 64 * MASK_WORDS;
constexpr int LUT_OFF = 20;          // LUT tick k sits at pair-word LUT_OFF + k of its zero-padded row
constexpr int SLAB_HDR = 4;          // slab header ints: bins, charge groups, first / last output block
constexpr int RESP_NO = 14;          // output ticks per response task (one thread: RESP_NO ticks x 2 target pixels)
constexpr int RESP_CONSUMERS = 256;  // consumer threads of the response kernel (8 warps, two per SM sub-partition)
constexpr int TILE_META = 4;         // ints per tile in lartpc_signals_t.tile_range: first / last output block, scale exponent, 0
constexpr int TC_TILE_BLOCK = 128;   // tiles per tensor-core tile block (MMA M of one CTA)
#ifndef LARTPC_CTA_PAIR
#define LARTPC_CTA_PAIR 0
#endif
constexpr bool TC_CTA_PAIR = LARTPC_CTA_PAIR != 0;  // the tensor-core response runs as CTA pairs (cta_group::2, M = 256 over two tile blocks)
constexpr int TC_UNIT_TILES = TC_CTA_PAIR ? 2 * TC_TILE_BLOCK : TC_TILE_BLOCK;   // tiles one response item multiplies at once:
                                     // the 16-tick block masks (tb_mask) are kept per unit

constexpr int SEG_REC_BYTES = 96, SEG_REC_BOX_OFFSET = 64;   // per-segment record of the tensor-core splat (charge_tc.cuh SegRec):
                                     // its last 32 bytes are the ints {N, a_lo, a_hi, b_lo, b_hi, jt0, jt1, flags}
constexpr int TC_BOXQ = 5;           // tile sort: classes per edge of the box of charged bins (bins 0-1, 2-3, .. 8-9 for 10 bins per pixel)
constexpr int TC_BOX_CLASSES = TC_BOXQ * TC_BOXQ * TC_BOXQ * TC_BOXQ;
constexpr int TC_CLASSES = 16 * TC_BOX_CLASSES;     // (16-tick block mask, box class)
constexpr int TC_CMASK_WORDS = 16;   // tc_cmask: per unit, 4 bits per LUT bin (the 16-tick blocks of that bin some tile of the unit
                                     // charges), 8 bins per 32-bit word, 128 operand rows

// device counters written by the planning kernels (mirrored to pinned host memory)
enum {
    CNT_MAX_NPIX = 0, CNT_MAX_TICKS, CNT_ACTIVE_SEGS, CNT_PAIRS, CNT_TILES, CNT_ACTIVE_PIX,
    CNT_TOTAL_SAMPLES, CNT_TOTAL_NPIX, CNT_OVERFLOW, CNT_COMPOSITE, CNT_CELLS, CNT_COUNT = 16
};

struct lartpc_sim {
    lartpc_params_t params;
    std::vector<lartpc_tpc_t> tpcs;
    DevParams dp;
    DevTpc *d_tpcs = nullptr;
    float *d_lut = nullptr;              // [NB2][WW][RS], zero padded rows
    std::vector<float> lut_copy;         // the table as given (host): source of the running-sum table of lartpc_hit_truth
    float *d_cum_lut = nullptr;          // [W nb][W nb][K] running sum over LUT ticks (built on the first lartpc_hit_truth)
    void *d_lut_tc = nullptr;            // tensor-core mode: fp16 hi / lo operand images of the LUT, [WW][NB2][2][NBW * 16]
    int64_t n_cp = 0;                    // charged-pixel grid cells over all TPCs
    int64_t n_pix = 0;                   // pixels over all TPCs (global pixel ids are 0 .. n_pix-1)
    int32_t pix_id_base = 0;
    // dense planning arrays
    int32_t *pix_count = nullptr, *pix_start = nullptr, *pix_tile0 = nullptr, *pix_cursor = nullptr;
    int32_t *pix_jmin = nullptr;         // first arrival tick on the charged pixel (window origin = this rounded down to a multiple of 4)
    unsigned long long *pix_mask = nullptr;   // [n_cp][MASK_WORDS] windows that hold charge
    int32_t *act_first = nullptr, *act_last = nullptr, *act_slot = nullptr;
    // growable planning arrays
    int32_t *pair_seg = nullptr;  int64_t pair_cap = 0;
    int32_t *tile_cp = nullptr;   TileDesc *tile_desc = nullptr;  int64_t tile_cap = 0;
    int32_t *cell_list = nullptr;        // [tile_cap] the charged cells that hold tiles, in no particular order (tile_emit_kernel)
    int2 *tile_list = nullptr;           // [tile_cap] {start, count} of the tile's segment list in pair_seg
    // tensor-core mode: tiles sorted by the 16-tick blocks they charge (launch_plan): slot of a tile, descriptors and
    // lists in slot order, per 128-slot block the OR of its tiles' block masks
    int32_t *tile_perm = nullptr;  TileDesc *tile_desc_p = nullptr;  int2 *tile_list_p = nullptr;
    int32_t *tb_mask = nullptr;  int32_t *cls_hist = nullptr;   // [tile_cap / 128 + 2], [2 TC_CLASSES]: class counts then cursors
    int32_t *tc_cmask = nullptr;         // [tile_cap / 128 + 2][TC_CMASK_WORDS]: blocks charged per (unit, bin), written by the charge lattice
    std::vector<int64_t> cp_base_h, pix_base_h;   // [n_tpcs + 1] first charged-pixel cell / first pixel of each TPC (host copy)
    int64_t plan_pix_lo = 0, plan_pix_hi = 0;       // pixel range of the TPCs the current plan covers
    int32_t *pack_base = nullptr, *pack_count = nullptr;  int pack_tile_pixels = 0;   // lartpc_pack_hits: readout-tile tables
    int64_t boxes_n = -1;  const void *boxes_of = nullptr;   // input whose S3 boxes the last tpc_lo = 0 plan wrote (reused by later batches)
    bool need_composite = false;         // some segment of the planned input wants composite node rules (charge_tc.cuh COMP)
    int batch_hint = 0;  size_t batch_hint_ws = 0;   // lartpc_run_spill: TPCs per batch that fitted the workspace last time
    void *seg_rec = nullptr;  int64_t seg_rec_cap = 0;   // per-segment records of the tensor-core splat (charge_tc.cuh)
    // scan scratch + counters
    long long *scan_tmp = nullptr;  int64_t scan_tmp_elems = 0;
    long long *d_counters = nullptr;  long long *h_counters = nullptr;
    uint32_t *disabled_mask = nullptr;
    int32_t *elec_slots = nullptr, *elec_offs = nullptr;  int64_t elec_slots_cap = 0, elec_offs_cap = 0;
    // plan state
    bool have_plan = false, have_signals = false;
    int64_t plan_n = 0, n_tiles = 0, n_pairs = 0, n_active = 0, total_samples = 0;
    const lartpc_drifted_t *plan_drifted = nullptr;
    lartpc_drifted_t drifted_copy;
    lartpc_pixmap_t pixmap_copy;
    int sm_count = 148;
    int device = 0;                      // CUDA device the sim was created on; every entry point runs there (DeviceGuard)
    // per-stage profiling of run_spill (lartpc_set_profiling)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_stage;           // stage of the event pair (2i, 2i+1)
    double stage_ms[LARTPC_N_STAGES] = {};
    int64_t stage_launches[LARTPC_N_STAGES] = {};
    double fma_current = 0.0;
    unsigned long long *d_fma = nullptr; // device counters of S4, LARTPC_N_COUNTERS of them ([0]: multiply-adds the method needs)
    double counters[8] = {};             // host copy after the last lartpc_run_spill (lartpc_get_counters)
    int *d_work = nullptr;               // work-queue cursor of the persistent response kernel
    int *d_end_row = nullptr;            // 16-byte row header with the END flag (terminates the consumers)
    unsigned char blk_of_slot[256];      // response kernel: output block of consumer-thread slot (balances the SM sub-partitions)
};

// ---- IEEE-exact float64 helpers (never contracted into FMA) -----------------------------------
__device__ __forceinline__ double xmul(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ double xadd(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ double xsub(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ double xdiv(double a, double b) { return __ddiv_rn(a, b); }
__device__ __forceinline__ double xsqrt(double a) { return __dsqrt_rn(a); }
__device__ __forceinline__ long long floor_div_ll(long long a, long long b)
{
    long long q = a / b;
    if ((a % b != 0) && ((a < 0) != (b < 0))) --q;
    return q;
}

// drift distance of a point, eq. (3.3): clamp(sign * (z - z_anode), 0, drift_len)
__device__ __forceinline__ double drift_dist(const DevTpc &t, double z)
{
    double d = xmul((double)t.sign, xsub(z, t.z_anode));
    if (d < 0.0) d = 0.0;
    if (d > t.drift_len) d = t.drift_len;
    return d;
}


// ---- Philox4x32-10 (Salmon et al., SC'11): counter (c0..c3), key (k0, k1) ----------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t lo0 = 0xD2511F53u * c0, hi0 = __umulhi(0xD2511F53u, c0);
        const uint32_t lo1 = 0xCD9E8D57u * c2, hi1 = __umulhi(0xCD9E8D57u, c2);
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}


// three standard normals of perturbed point (segment s, mu, nu) of eq. (3.9) as printed (reading D25): Box-Muller pairs
// of Philox(counter (s, mu, nu, 'RAND'), key = seed), clamped to +- clamp
__device__ __forceinline__ void perturbation_normals(unsigned long long seed, uint32_t s, uint32_t mu, uint32_t nu,
                                                     double clamp, double (&z)[3])
{
    uint32_t x[4];
    philox4x32_10(s, mu, nu, 0x52414E44u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
    const double sc = 1.0 / 4294967296.0, two_pi = 6.283185307179586476925286766559;
    const double u0 = ((double)x[0] + 0.5) * sc, u1 = ((double)x[1] + 0.5) * sc;
    const double u2 = ((double)x[2] + 0.5) * sc, u3 = ((double)x[3] + 0.5) * sc;
    const double r01 = sqrt(-2.0 * log(u0)), r23 = sqrt(-2.0 * log(u2));
    z[0] = r01 * cos(two_pi * u1);
    z[1] = r01 * sin(two_pi * u1);
    z[2] = r23 * cos(two_pi * u3);
#pragma unroll
    for (int k = 0; k < 3; ++k) z[k] = fmin(fmax(z[k], -clamp), clamp);
}

// ---- launch helpers -----------------------------------------------------------------------------
static inline int div_up(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// The charge lattice runs on the tensor cores (charge_tc.cuh) when the response does and the bins of a pixel fill one
// 128-row operand the kernel is instantiated for; otherwise the FFMA2 splat writes the same operand image in the
// tiles' original order.  ONE predicate for the plan (tile sort), the per-segment records and the splat dispatch.
static inline bool splat_on_tc(const DevParams &p) { return p.tc_mode && (p.nb == 10 || p.nb == 5); }

// cudaFuncAttributeMaxDynamicSharedMemorySize is per device: remember, per kernel and device, what has been set
constexpr int LARTPC_MAX_DEVICES = 64;
struct SmemCfg { size_t bytes[LARTPC_MAX_DEVICES] = {}; };
template <typename F> static inline cudaError_t ensure_dyn_smem(F func, SmemCfg &cfg, int device, size_t bytes)
{
    if (device < 0 || device >= LARTPC_MAX_DEVICES) return cudaErrorInvalidDevice;
    if (bytes <= cfg.bytes[device]) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e == cudaSuccess) cfg.bytes[device] = bytes;
    return e;
}

// entry points run on the sim's device whatever the caller's current device is, and restore it
struct DeviceGuard {
    int prev = -1;  bool switched = false;
    explicit DeviceGuard(int device)
    {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != device) switched = cudaSetDevice(device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// stage launchers (host, C++ linkage)
int launch_quench(lartpc_sim *sim, const lartpc_segments_t *seg, int64_t n, float *dEdx, float *n_e, cudaStream_t st);
int launch_drift(lartpc_sim *sim, const lartpc_segments_t *seg, int64_t n, const float *n_e, lartpc_drifted_t *out,
                 cudaStream_t st);
int sim_grow_tiles(lartpc_sim *sim, int64_t cap);
int launch_plan(lartpc_sim *sim, const lartpc_segments_t *seg, const lartpc_drifted_t *dr, int64_t n,
                int tpc_lo, int tpc_hi, lartpc_pixmap_t *out, lartpc_pixmap_info_t *info, cudaStream_t st);
int launch_current_splat(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n,
                         lartpc_signals_t *out, cudaStream_t st);
int launch_hit_truth(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, const lartpc_hits_t *hits,
                     int64_t n_hits, lartpc_truth_t *out, cudaStream_t st);
int launch_seg_records(lartpc_sim *sim, const lartpc_drifted_t *dr, const lartpc_pixmap_t *pm, int64_t n, cudaStream_t st);
int launch_current_response(lartpc_sim *sim, lartpc_signals_t *out, cudaStream_t st);
int launch_current_response_tc(lartpc_sim *sim, lartpc_signals_t *out, cudaStream_t st);
size_t lartpc_build_lut_tc(const DevParams &p, const float *lut_host, void **d_out);   // returns bytes, 0 on failure
static inline int64_t tiles_alloc(const DevParams &p, int64_t n_tiles)
{
    return p.tc_mode ? (n_tiles + TC_UNIT_TILES - 1) / TC_UNIT_TILES * TC_UNIT_TILES : n_tiles;
}
int launch_pack_hits(lartpc_sim *sim, const lartpc_hits_t *hits, int64_t n_hits, int tile_pixels, uint16_t *packed,
                     int64_t *tile_offsets, cudaStream_t st);
int launch_sum(lartpc_sim *sim, const lartpc_signals_t *sig, lartpc_waveforms_t *out, cudaStream_t st);
int static_scratch_ptr(int device, void **ptr);   // stages_pixel.cu: device address of lartpc_electronics_static's scratch (device current)
int launch_electronics(lartpc_sim *sim, const lartpc_waveforms_t *wf, uint64_t seed, lartpc_hits_t *out,
                       int32_t *slot_scratch, int32_t *scan_scratch, int64_t hit_base, cudaStream_t st);
int sim_ensure_scan_tmp(lartpc_sim *sim, int64_t elems);
