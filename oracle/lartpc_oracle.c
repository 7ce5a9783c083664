/*
 * lartpc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, fp64 CPU statement of the charge-readout hot path of arXiv 2212.09807
 * ("Highly-parallelized simulation of a pixelated LArTPC on a GPU"), written from the paper
 * (/root/reference/PAPER.md, cited as P:L###) and the readings D1-D23 listed in DESIGN.md.
 * It shares no code, header, table or helper with the CUDA library; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC lartpc_oracle.c -lm
 *        (-ffp-contract=off: every integer decision below must come from individually rounded
 *         IEEE-754 double operations, in the order written.)
 *
 * Parity pins (tests/test_oracle_pins.py, all "-m 'not gpu'"); every function AND branch below has one:
 *   orc_quench      Birks / Box branches: closed forms eqs. (3.1)(3.2) (test_recombination_golden_values, printed "around
 *                   0.7" for a MIP), invariants (1/R linear; exp(R xi) - xi = alpha); R < 0 clamp, L = 0, dE = 0
 *                   (test_recombination_invariants)
 *   orc_drift       exp(-t/tau), sigma = sqrt(2 D t) values (test_transport_golden_values); sign of eq. (3.3) for
 *                   two-sided modules and the inactive branch (test_drift_two_sided_module_and_inactive)
 *   orc_pixmap      hand-worked rectangles at sigma = 0 and at the plane edge (test_pixmap_hand_cases); charged-bin box
 *                   and tick range jt0 / jt1 with sigma > 0 and t_origin != 0 (test_pixmap_tick_range_with_diffusion);
 *                   brute-force completeness / minimality (test_pixmap_complete_and_minimal)
 *   orc_pixel_current  zero-diffusion point charge == LUT (sigma = 0 indicator branch), charge conservation, long-track
 *                   erf closed form, per-electron Monte Carlo, direct 6-fold sum (orc_direct_current)
 *   orc_pixel_current_random  (eq. 3.9 as printed) exact charge conservation, sigma = 0 identity with the
 *                   expectation form, one perturbed point placed by hand, mean over seeds vs the expectation form
 *   orc_philox4x32_10 / orc_noise_normals   Random123 known answers; moments; the test's own pure-Python Philox +
 *                   Box-Muller reproduces the three normals (test_python_philox_matches_the_published_vectors)
 *   orc_electronics branch by branch, expected ticks / counts worked in the test from its own Philox normals:
 *                   integrate / threshold (>=) / hold / ADC floor + clamp / window end   test_electronics_hand_cases
 *                   reset noise q = noise_reset * z_r after the sample                    test_electronics_reset_noise_branch
 *                   uncorrelated noise on the sampled value (z_u)                         test_electronics_uncorrelated_noise_branch
 *                   discriminator noise on the threshold, fresh each tick (z_d)           test_electronics_discriminator_noise_branch
 *                   periodic reset (armed only, before the tick's charge)                 test_electronics_periodic_reset_branch
 *                   min-spacing re-arm (n >= sample + spacing - hold)                     test_electronics_min_spacing_branch
 *   orc_segment_currents / orc_hit_truth  (O7, truth association)  three point charges placed by hand under a delta-like
 *                   LUT: shares, fractions and window starts written out in the test (test_hit_truth_hand_case); the
 *                   periodic-reset window start (test_hit_truth_periodic_reset_window); shares of all segments add up to the
 *                   integral of orc_pixel_current's waveform over the window, and that integral reproduces the noise-free
 *                   ADC code of orc_electronics (test_hit_truth_sums_to_the_sampled_charge)
 *   Light simulation (NEXT-3; tests/test_oracle_light_pins.py):
 *   orc_light_npe             photon yield worked by hand from eqs. (3.2)(4.1), voxel / tick indices and the outside-the-grid
 *                             branch by hand, N_gamma + n_e = dE / W_ph (test_light_photon_yield_and_voxels_by_hand)
 *   orc_light_profile         hand-placed segments with lut_m = 2, light past the waveform dropped, conservation
 *   orc_light_scint_weights   closed forms of the tick-integrated eq. (4.4), telescoping sum > 0.99, first-order
 *                             agreement with f_scint(s dt) dt as eq. (4.5) prints it
 *   orc_light_convolve        numpy.convolve, impulse, steady state
 *   orc_light_fluctuate(_one) scipy.stats.poisson.ppf at the test's own Philox uniform (Poisson branch), Box-Muller by hand
 *                             (normal branch), lambda <= 0, moments
 *   orc_light_noise           one sensor's sinusoids by hand from the Philox phase, mean square
 *   (whole chain: test_light_chain_conserves_light)
 *   No function is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif
/* threads of the pixel loops (orc_plane_currents*); no arithmetic here.  Returns the count in effect. */
int orc_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
    return omp_get_max_threads();
#else
    (void)n;
    return 1;
#endif
}

typedef struct {
    double e_field, rho, w_ion;              /* kV/cm, g/cm^3, MeV per electron */
    int    recomb_model;                     /* 0 Birks eq. (3.1), 1 modified Box eq. (3.2) */
    double birks_ab, birks_kb, box_alpha, box_beta;
    double v_drift, lifetime, d_long, d_tran; /* cm/us, us, cm^2/us, cm^2/us */
    double dt, t_origin;                     /* us */
    double pitch;                            /* cm */
    int    nb, wpix, klut, n_ticks;          /* bins per pixel, window pixels, LUT ticks, readout ticks */
    double sample_step, n_sigma_map;         /* cm, - */
    double gain_mv_per_ke, v_cm, v_ref, v_ped; int adc_bits;
    double threshold_e; int hold_ticks, min_spacing_ticks, periodic_reset_ticks;
    double noise_reset_e, noise_disc_e, noise_uncorr_e;
    int    max_hits_per_pixel;
} orc_params;

typedef struct { double x0, y0, z_anode; int drift_sign; double drift_len; int nx, ny, first_pixel_id; } orc_tpc;

/* ---------------------------------------------------------------------------------------------
 * O1  Electron recombination.  Q_R = R * Q_0, Q_0 = dE / W_ion.
 *   Birks  R = A_b / (1 + k_b/eps * dE/dx)                 eq. (3.1)
 *   Box    R = ln(alpha + beta/eps * dE/dx) / (beta/eps * dE/dx)   eq. (3.2), clamped >= 0 (D6)
 *   eps = E * rho.  R is a fixed number, no fluctuation.
 * ------------------------------------------------------------------------------------------- */
void orc_quench(const orc_params *p, int64_t n,
                const float *xs, const float *ys, const float *zs,
                const float *xe, const float *ye, const float *ze, const float *dE,
                double *dEdx, double *n_e)
{
    const double eps = p->e_field * p->rho;
    for (int64_t i = 0; i < n; ++i) {
        double dx = (double)xe[i] - (double)xs[i];
        double dy = (double)ye[i] - (double)ys[i];
        double dz = (double)ze[i] - (double)zs[i];
        double L = sqrt((dx * dx + dy * dy) + dz * dz);
        double e = (double)dE[i];
        if (!(L > 0.0) || !(e > 0.0)) { dEdx[i] = 0.0; n_e[i] = 0.0; continue; }
        double q = e / L;                                   /* dE/dx, MeV/cm */
        double R;
        if (p->recomb_model == 0) {
            R = p->birks_ab / (1.0 + p->birks_kb * q / eps);
        } else {
            double xi = p->box_beta * q / eps;
            R = log(p->box_alpha + xi) / xi;
            if (R < 0.0) R = 0.0;
        }
        dEdx[i] = q;
        n_e[i] = R * (e / p->w_ion);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O2  Electron transport.
 *   TPC = first one whose box holds the segment midpoint, else inactive (D8).
 *   drift distance d(z) = clamp(sign*(z - z_anode), 0, drift_len); t_drift = d / v_drift  eq. (3.3)
 *   Q_a = Q_R exp(-t_drift/tau)                                                       eq. (3.4)
 *   sigma = sqrt(2 D t_drift), D_L and D_T                                             eq. (3.5)
 *   one value per segment, taken at the midpoint (D9); sigma_t = sigma_L / v_drift.
 *   Arrival times of the two ends T = t + d(z)/v_drift; plane-local u = x - x0, v = y - y0.
 * ------------------------------------------------------------------------------------------- */
static double drift_dist(const orc_tpc *t, double z)
{
    double d = (double)t->drift_sign * (z - t->z_anode);
    if (d < 0.0) d = 0.0;
    if (d > t->drift_len) d = t->drift_len;
    return d;
}

void orc_drift(const orc_params *p, const orc_tpc *tpcs, int n_tpcs, int64_t n,
               const float *xs, const float *ys, const float *zs, const float *ts,
               const float *xe, const float *ye, const float *ze, const float *te,
               const double *n_e,
               int32_t *tpc, double *q_a, double *sigma_T, double *sigma_t,
               double *u_s, double *v_s, double *u_e, double *v_e, double *T_s, double *T_e)
{
    for (int64_t i = 0; i < n; ++i) {
        double xm = 0.5 * ((double)xs[i] + (double)xe[i]);
        double ym = 0.5 * ((double)ys[i] + (double)ye[i]);
        double zm = 0.5 * ((double)zs[i] + (double)ze[i]);
        int found = -1;
        for (int k = 0; k < n_tpcs && found < 0; ++k) {
            const orc_tpc *t = &tpcs[k];
            double x1 = t->x0 + (double)t->nx * p->pitch;
            double y1 = t->y0 + (double)t->ny * p->pitch;
            double dm = (double)t->drift_sign * (zm - t->z_anode);
            if (xm >= t->x0 && xm < x1 && ym >= t->y0 && ym < y1 && dm >= 0.0 && dm <= t->drift_len) found = k;
        }
        tpc[i] = found;
        if (found < 0) {
            q_a[i] = sigma_T[i] = sigma_t[i] = 0.0;
            u_s[i] = v_s[i] = u_e[i] = v_e[i] = T_s[i] = T_e[i] = 0.0;
            continue;
        }
        const orc_tpc *t = &tpcs[found];
        double t_mid = drift_dist(t, zm) / p->v_drift;
        q_a[i] = n_e[i] * exp(-t_mid / p->lifetime);
        sigma_T[i] = sqrt((2.0 * p->d_tran) * t_mid);
        double sigma_L = sqrt((2.0 * p->d_long) * t_mid);
        sigma_t[i] = sigma_L / p->v_drift;
        u_s[i] = (double)xs[i] - t->x0;  v_s[i] = (double)ys[i] - t->y0;
        u_e[i] = (double)xe[i] - t->x0;  v_e[i] = (double)ye[i] - t->y0;
        T_s[i] = (double)ts[i] + drift_dist(t, (double)zs[i]) / p->v_drift;
        T_e[i] = (double)te[i] + drift_dist(t, (double)ze[i]) / p->v_drift;
    }
}

/* ---------------------------------------------------------------------------------------------
 * O3  Pixel mapping ("the length of the longest signal and the largest number of pixels
 *     per segment are calculated before execution"; P:L695 neighbours get signal through
 *     transverse diffusion).  The algorithm is not in the paper: reading D10.
 *   charged-bin range  a_lo = floor((min(u_s,u_e) - r)/bin), a_hi = floor((max(u_s,u_e) + r)/bin),
 *                      r = n_sigma_map * sigma_T, bin = pitch/nb; same in v;
 *   pixel rectangle    [floor_div(a_lo,nb) - H, floor_div(a_hi,nb) + H] clipped to the plane, H=(W-1)/2;
 *   arrival ticks      jt0 = floor(((min(T) - rt) - t_origin)/dt), jt1 with max and +, rt = n_sigma_map*sigma_t;
 *   samples            N = max(1, ceil(L / sample_step))  (D3).
 * ------------------------------------------------------------------------------------------- */
static int64_t floor_div(int64_t a, int64_t b) { int64_t q = a / b; if ((a % b != 0) && ((a < 0) != (b < 0))) --q; return q; }

void orc_pixmap(const orc_params *p, const orc_tpc *tpcs, int64_t n,
                const float *xs, const float *ys, const float *zs,
                const float *xe, const float *ye, const float *ze,
                const int32_t *tpc, const double *q_a, const double *sigma_T, const double *sigma_t,
                const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                const double *T_s, const double *T_e,
                int32_t *a_lo, int32_t *a_hi, int32_t *b_lo, int32_t *b_hi,
                int32_t *ix0, int32_t *ix1, int32_t *iy0, int32_t *iy1,
                int32_t *jt0, int32_t *jt1, int32_t *npix, int32_t *n_samples)
{
    const double bin = p->pitch / (double)p->nb;
    const int H = (p->wpix - 1) / 2;
    for (int64_t i = 0; i < n; ++i) {
        double dx = (double)xe[i] - (double)xs[i];
        double dy = (double)ye[i] - (double)ys[i];
        double dz = (double)ze[i] - (double)zs[i];
        double L = sqrt((dx * dx + dy * dy) + dz * dz);
        int64_t N = (int64_t)ceil(L / p->sample_step);
        if (N < 1) N = 1;
        n_samples[i] = (int32_t)N;
        if (tpc[i] < 0 || !(q_a[i] > 0.0)) {
            a_lo[i] = b_lo[i] = 0; a_hi[i] = b_hi[i] = -1;
            ix0[i] = iy0[i] = 0; ix1[i] = iy1[i] = -1; jt0[i] = 0; jt1[i] = -1; npix[i] = 0;
            continue;
        }
        const orc_tpc *t = &tpcs[tpc[i]];
        double r = p->n_sigma_map * sigma_T[i];
        double umin = fmin(u_s[i], u_e[i]), umax = fmax(u_s[i], u_e[i]);
        double vmin = fmin(v_s[i], v_e[i]), vmax = fmax(v_s[i], v_e[i]);
        int64_t al = (int64_t)floor((umin - r) / bin), ah = (int64_t)floor((umax + r) / bin);
        int64_t bl = (int64_t)floor((vmin - r) / bin), bh = (int64_t)floor((vmax + r) / bin);
        a_lo[i] = (int32_t)al; a_hi[i] = (int32_t)ah; b_lo[i] = (int32_t)bl; b_hi[i] = (int32_t)bh;
        int64_t x0 = floor_div(al, p->nb) - H, x1 = floor_div(ah, p->nb) + H;
        int64_t y0 = floor_div(bl, p->nb) - H, y1 = floor_div(bh, p->nb) + H;
        if (x0 < 0) x0 = 0;
        if (y0 < 0) y0 = 0;
        if (x1 > t->nx - 1) x1 = t->nx - 1;
        if (y1 > t->ny - 1) y1 = t->ny - 1;
        ix0[i] = (int32_t)x0; ix1[i] = (int32_t)x1; iy0[i] = (int32_t)y0; iy1[i] = (int32_t)y1;
        npix[i] = (x0 <= x1 && y0 <= y1) ? (int32_t)((x1 - x0 + 1) * (y1 - y0 + 1)) : 0;
        double rt = p->n_sigma_map * sigma_t[i];
        double tmin = fmin(T_s[i], T_e[i]), tmax = fmax(T_s[i], T_e[i]);
        jt0[i] = (int32_t)floor(((tmin - rt) - p->t_origin) / p->dt);
        jt1[i] = (int32_t)floor(((tmax + rt) - p->t_origin) / p->dt);
    }
}

/* ---------------------------------------------------------------------------------------------
 * O4 + O5  Induced current on ONE pixel, summed over segments.
 *
 *   eq. (3.7)  I(t) = Int I_pixel(t - z/v_d, x, y) rho(x,y,z) dx dy dz
 *   eq. (3.8)  rho ~ Q_a/(N M) sum_mu sum_nu delta(x_mu + dx_mu_nu - x) ...   (N points, M perturbations)
 *   eq. (3.9)  I(t) ~ Q_a/(N M) sum_mu sum_nu I_pixel(t - (z_mu+dz)/v_d, x_mu+dx, y_mu+dy)
 *
 *   Reading D1: the M-sum is taken in expectation (its M -> infinity limit).  Reading D3: the N points
 *   are the regular midpoints f = (mu + 1/2)/N, N from a 10 um interval.  Reading D4: the LUT
 *   is piecewise constant over (x, y) bins of size `bin` and over ticks ("discrete (x,y) locations ...
 *   discrete time"), so the expectation of the Gaussian perturbation over one LUT cell is the
 *   product of three normal-CDF differences.  Reading D5: LUT tick K-1 is the arrival tick; an electron
 *   arriving in arrival tick j contributes R[cy][cx][k] to readout tick n = j + k.
 *
 *   Written out in the paper's order: first rho integrated over every LUT cell of this pixel's
 *   W x W-pixel window (eq. 3.8 in expectation) -> G[cy][cx][j]; then eq. (3.7) as the finite sum
 *   I_p[n] = sum_{cy,cx} sum_j G[cy][cx][j] * R[cy][cx][n-j].
 *   Charge arriving outside arrival ticks [0, n_ticks - K] is outside the readout window (D23).
 *   There is no truncation parameter: a segment is skipped for a pixel only when every cell of the
 *   window is farther than 9 sigma from its bounding box (weights below 1e-18).
 *
 *   Segment arrays are those of orc_drift / orc_pixmap; only segments with tpc[i] == tpc_index count.
 *   wave[n_ticks] is overwritten.  Returns the sum of wave (Q_p, O5).
 * ------------------------------------------------------------------------------------------- */
static double phi_cdf(double x) { return 0.5 * erfc(-x * 0.70710678118654752440); }

/* weight of the interval [lo, hi) under N(mean, sigma); sigma == 0 -> indicator (D4) */
static double cell_weight(double lo, double hi, double mean, double sigma)
{
    return phi_cdf((hi - mean) / sigma) - phi_cdf((lo - mean) / sigma);
}

double orc_pixel_current(const orc_params *p, const orc_tpc *tpcs, int tpc_index, const float *lut,
                         int64_t n, const int32_t *tpc, const double *q_a,
                         const double *sigma_T, const double *sigma_t,
                         const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                         const double *T_s, const double *T_e, const int32_t *n_samples,
                         int ix, int iy, double *wave)
{
    (void)tpcs;
    const int nb = p->nb, W = p->wpix, K = p->klut, H = (W - 1) / 2, NB = W * nb;
    const double bin = p->pitch / (double)nb;
    const int64_t j_max = (int64_t)p->n_ticks - K;              /* last arrival tick inside the window */
    const int64_t a_org = (int64_t)nb * (ix - H), b_org = (int64_t)nb * (iy - H);  /* first bin of the window */
    memset(wave, 0, sizeof(double) * (size_t)p->n_ticks);
    if (j_max < 0) return 0.0;
    const size_t nj = (size_t)(j_max + 1);
    double *G = (double *)calloc((size_t)NB * NB * nj, sizeof(double));
    double *wx = (double *)malloc(sizeof(double) * NB), *wy = (double *)malloc(sizeof(double) * NB);
    double *wt = (double *)malloc(sizeof(double) * nj);
    int64_t jlo_used = j_max + 1, jhi_used = -1;
    for (int64_t s = 0; s < n; ++s) {
        if (tpc[s] != tpc_index || !(q_a[s] > 0.0)) continue;
        const double sT = sigma_T[s], st = sigma_t[s];
        /* skip when the whole window is > 9 sigma away from the segment's bounding box */
        double reach = 9.0 * sT;
        double ulo = fmin(u_s[s], u_e[s]) - reach, uhi = fmax(u_s[s], u_e[s]) + reach;
        double vlo = fmin(v_s[s], v_e[s]) - reach, vhi = fmax(v_s[s], v_e[s]) + reach;
        if (uhi < (double)a_org * bin || ulo > (double)(a_org + NB) * bin) continue;
        if (vhi < (double)b_org * bin || vlo > (double)(b_org + NB) * bin) continue;
        const int N = n_samples[s];
        const double q = q_a[s] / (double)N;                     /* eq. (3.8): Q_a / N per point */
        for (int mu = 0; mu < N; ++mu) {
            double f = ((double)mu + 0.5) / (double)N;
            double u = u_s[s] + (u_e[s] - u_s[s]) * f;
            double v = v_s[s] + (v_e[s] - v_s[s]) * f;
            double T = T_s[s] + (T_e[s] - T_s[s]) * f;
            int cx0 = NB, cx1 = -1, cy0 = NB, cy1 = -1; int64_t j0 = j_max + 1, j1 = -1;
            if (sT > 0.0) {
                /* bins farther than 9 sigma from the point carry < 1e-18 of its charge */
                for (int c = 0; c < NB; ++c) {
                    double x_lo = (double)(a_org + c) * bin, x_hi = (double)(a_org + c + 1) * bin;
                    double y_lo = (double)(b_org + c) * bin, y_hi = (double)(b_org + c + 1) * bin;
                    wx[c] = (x_hi < u - reach || x_lo > u + reach) ? 0.0 : cell_weight(x_lo, x_hi, u, sT);
                    wy[c] = (y_hi < v - reach || y_lo > v + reach) ? 0.0 : cell_weight(y_lo, y_hi, v, sT);
                    if (wx[c] > 0.0) { if (c < cx0) cx0 = c; cx1 = c; }
                    if (wy[c] > 0.0) { if (c < cy0) cy0 = c; cy1 = c; }
                }
            } else {
                for (int c = 0; c < NB; ++c) wx[c] = wy[c] = 0.0;
                int64_t a = (int64_t)floor(u / bin) - a_org, b = (int64_t)floor(v / bin) - b_org;
                if (a >= 0 && a < NB) { wx[a] = 1.0; cx0 = cx1 = (int)a; }
                if (b >= 0 && b < NB) { wy[b] = 1.0; cy0 = cy1 = (int)b; }
            }
            if (cx1 < 0 || cy1 < 0) continue;
            if (st > 0.0) {
                int64_t ja = (int64_t)floor(((T - 9.0 * st) - p->t_origin) / p->dt);
                int64_t jb = (int64_t)floor(((T + 9.0 * st) - p->t_origin) / p->dt);
                if (ja < 0) ja = 0;
                if (jb > j_max) jb = j_max;
                for (int64_t j = ja; j <= jb; ++j) {
                    double t_lo = p->t_origin + (double)j * p->dt, t_hi = p->t_origin + (double)(j + 1) * p->dt;
                    wt[j] = cell_weight(t_lo, t_hi, T, st);
                }
                j0 = ja; j1 = jb;
            } else {
                int64_t j = (int64_t)floor((T - p->t_origin) / p->dt);
                if (j >= 0 && j <= j_max) { wt[j] = 1.0; j0 = j1 = j; }
            }
            if (j1 < j0) continue;
            if (j0 < jlo_used) jlo_used = j0;
            if (j1 > jhi_used) jhi_used = j1;
            for (int cy = cy0; cy <= cy1; ++cy)
                for (int cx = cx0; cx <= cx1; ++cx) {
                    double wxy = q * wy[cy] * wx[cx];
                    double *g = G + ((size_t)cy * NB + cx) * nj;
                    for (int64_t j = j0; j <= j1; ++j) g[j] += wxy * wt[j];
                }
        }
    }
    /* eq. (3.7) on the lattice: I_p[n] = sum_cells G * R, n = j + k */
    double total = 0.0;
    if (jhi_used >= jlo_used) {
        for (int cy = 0; cy < NB; ++cy)
            for (int cx = 0; cx < NB; ++cx) {
                const double *g = G + ((size_t)cy * NB + cx) * nj;
                const float *r = lut + ((size_t)cy * NB + cx) * K;
                for (int64_t j = jlo_used; j <= jhi_used; ++j) {
                    double c = g[j];
                    if (c == 0.0) continue;
                    for (int k = 0; k < K; ++k) wave[j + k] += c * (double)r[k];
                }
            }
        for (int nidx = 0; nidx < p->n_ticks; ++nidx) total += wave[nidx];
    }
    free(G); free(wx); free(wy); free(wt);
    return total;
}

/* Many pixels of one TPC (row-major list of (ix, iy) pairs); waves[npx][n_ticks], q_p[npx].
 * Pixels are independent, so this loop may run on several threads (-fopenmp). */
void orc_plane_currents(const orc_params *p, const orc_tpc *tpcs, int tpc_index, const float *lut,
                        int64_t n, const int32_t *tpc, const double *q_a,
                        const double *sigma_T, const double *sigma_t,
                        const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                        const double *T_s, const double *T_e, const int32_t *n_samples,
                        int64_t npx, const int32_t *ixs, const int32_t *iys, double *waves, double *q_p)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < npx; ++k)
        q_p[k] = orc_pixel_current(p, tpcs, tpc_index, lut, n, tpc, q_a, sigma_T, sigma_t,
                                   u_s, v_s, u_e, v_e, T_s, T_e, n_samples,
                                   ixs[k], iys[k], waves + (size_t)k * p->n_ticks);
}

/* ---------------------------------------------------------------------------------------------
 * O4r  Eq. (3.9) as printed: every one of the N points of a segment is perturbed M times,
 *   I(t) ~ Q_a/(N M) sum_mu sum_nu I_pixel(t - (z_mu + dz_mu_nu)/v_d, x_mu + dx_mu_nu, y_mu + dy_mu_nu),
 * with (dx, dy) ~ N(0, sigma_T), dz/v_d ~ N(0, sigma_t).  Reading D25: the normals of point
 * (segment s, mu, nu) are Box-Muller pairs of Philox4x32-10(counter = (s, mu, nu, 0x52414E44), key = seed):
 * z1 = r01 cos, z2 = r01 sin, z3 = r23 cos, u_i = (x_i + 0.5) 2^-32, each clamped to +- n_sigma_map so that every
 * perturbed point stays inside the rectangle and tick range O3 gives the segment.  The look-up is nearest-bin in
 * x, y and t (D4), so a perturbed point adds Q_a/(N M) to exactly one LUT cell.  s is the index in the arrays
 * passed in.  Same lattice-then-convolution order as orc_pixel_current.
 * ------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

void orc_perturbation_normals(uint64_t seed, uint32_t s, uint32_t mu, uint32_t nu, double clamp, double z[3])
{
    uint32_t ctr[4] = { s, mu, nu, 0x52414E44u }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
    orc_philox4x32_10(ctr, key, x);
    const double two_pi = 6.283185307179586476925286766559;
    double u0 = ((double)x[0] + 0.5) * (1.0 / 4294967296.0), u1 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
    double u2 = ((double)x[2] + 0.5) * (1.0 / 4294967296.0), u3 = ((double)x[3] + 0.5) * (1.0 / 4294967296.0);
    double r01 = sqrt(-2.0 * log(u0)), r23 = sqrt(-2.0 * log(u2));
    z[0] = r01 * cos(two_pi * u1);
    z[1] = r01 * sin(two_pi * u1);
    z[2] = r23 * cos(two_pi * u3);
    for (int k = 0; k < 3; ++k) { if (z[k] > clamp) z[k] = clamp; if (z[k] < -clamp) z[k] = -clamp; }
}

double orc_pixel_current_random(const orc_params *p, int tpc_index, const float *lut,
                                int64_t n, const int32_t *tpc, const double *q_a,
                                const double *sigma_T, const double *sigma_t,
                                const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                                const double *T_s, const double *T_e, const int32_t *n_samples,
                                int M, uint64_t seed, int ix, int iy, double *wave)
{
    const int nb = p->nb, W = p->wpix, K = p->klut, H = (W - 1) / 2, NB = W * nb;
    const double bin = p->pitch / (double)nb;
    const int64_t j_max = (int64_t)p->n_ticks - K;
    const int64_t a_org = (int64_t)nb * (ix - H), b_org = (int64_t)nb * (iy - H);
    memset(wave, 0, sizeof(double) * (size_t)p->n_ticks);
    if (j_max < 0 || M < 1) return 0.0;
    const size_t nj = (size_t)(j_max + 1);
    double *G = (double *)calloc((size_t)NB * NB * nj, sizeof(double));
    int64_t jlo_used = j_max + 1, jhi_used = -1;
    for (int64_t s = 0; s < n; ++s) {
        if (tpc[s] != tpc_index || !(q_a[s] > 0.0)) continue;
        const double sT = sigma_T[s], st = sigma_t[s], reach = p->n_sigma_map * sT;
        if (fmax(u_s[s], u_e[s]) + reach < (double)a_org * bin || fmin(u_s[s], u_e[s]) - reach > (double)(a_org + NB) * bin) continue;
        if (fmax(v_s[s], v_e[s]) + reach < (double)b_org * bin || fmin(v_s[s], v_e[s]) - reach > (double)(b_org + NB) * bin) continue;
        const int N = n_samples[s];
        const double q = q_a[s] / (double)N / (double)M;          /* eq. (3.9): Q_a / (N M) per perturbed point */
        for (int mu = 0; mu < N; ++mu) {
            double f = ((double)mu + 0.5) / (double)N;
            double u = u_s[s] + (u_e[s] - u_s[s]) * f;
            double v = v_s[s] + (v_e[s] - v_s[s]) * f;
            double T = T_s[s] + (T_e[s] - T_s[s]) * f;
            for (int nu = 0; nu < M; ++nu) {
                double z[3];
                orc_perturbation_normals(seed, (uint32_t)s, (uint32_t)mu, (uint32_t)nu, p->n_sigma_map, z);
                double uu = u + sT * z[0], vv = v + sT * z[1], TT = T + st * z[2];
                int64_t a = (int64_t)floor(uu / bin) - a_org, b = (int64_t)floor(vv / bin) - b_org;
                int64_t j = (int64_t)floor((TT - p->t_origin) / p->dt);
                if (a < 0 || a >= NB || b < 0 || b >= NB || j < 0 || j > j_max) continue;
                G[((size_t)b * NB + (size_t)a) * nj + (size_t)j] += q;
                if (j < jlo_used) jlo_used = j;
                if (j > jhi_used) jhi_used = j;
            }
        }
    }
    double total = 0.0;
    if (jhi_used >= jlo_used) {
        for (int cy = 0; cy < NB; ++cy)
            for (int cx = 0; cx < NB; ++cx) {
                const double *g = G + ((size_t)cy * NB + cx) * nj;
                const float *r = lut + ((size_t)cy * NB + cx) * K;
                for (int64_t j = jlo_used; j <= jhi_used; ++j) {
                    double c = g[j];
                    if (c == 0.0) continue;
                    for (int k = 0; k < K; ++k) wave[j + k] += c * (double)r[k];
                }
            }
        for (int nidx = 0; nidx < p->n_ticks; ++nidx) total += wave[nidx];
    }
    free(G);
    return total;
}

void orc_plane_currents_random(const orc_params *p, int tpc_index, const float *lut,
                               int64_t n, const int32_t *tpc, const double *q_a,
                               const double *sigma_T, const double *sigma_t,
                               const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                               const double *T_s, const double *T_e, const int32_t *n_samples,
                               int M, uint64_t seed,
                               int64_t npx, const int32_t *ixs, const int32_t *iys, double *waves, double *q_p)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < npx; ++k)
        q_p[k] = orc_pixel_current_random(p, tpc_index, lut, n, tpc, q_a, sigma_T, sigma_t, u_s, v_s, u_e, v_e,
                                          T_s, T_e, n_samples, M, seed, ixs[k], iys[k],
                                          waves + (size_t)k * p->n_ticks);
}

/* The same quantity as the literal nested sum of SURVEY.md 8(c.1), one term at a time and without the
 * intermediate lattice (tiny inputs only; pins orc_pixel_current against a reordering mistake):
 *   I_p[n] = sum_seg sum_mu (Q_a/N) sum_a sum_b sum_j wx[a] wy[b] wt[j] R[b - nb(iy-H)][a - nb(ix-H)][n - j] */
void orc_direct_current(const orc_params *p, int tpc_index, const float *lut,
                        int64_t n, const int32_t *tpc, const double *q_a,
                        const double *sigma_T, const double *sigma_t,
                        const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                        const double *T_s, const double *T_e, const int32_t *n_samples,
                        int ix, int iy, double *wave)
{
    const int nb = p->nb, W = p->wpix, K = p->klut, H = (W - 1) / 2, NB = W * nb;
    const double bin = p->pitch / (double)nb;
    const int64_t j_max = (int64_t)p->n_ticks - K;
    for (int nidx = 0; nidx < p->n_ticks; ++nidx) {
        double acc = 0.0;
        for (int64_t s = 0; s < n; ++s) {
            if (tpc[s] != tpc_index || !(q_a[s] > 0.0)) continue;
            const int N = n_samples[s];
            for (int mu = 0; mu < N; ++mu) {
                double f = ((double)mu + 0.5) / (double)N;
                double u = u_s[s] + (u_e[s] - u_s[s]) * f;
                double v = v_s[s] + (v_e[s] - v_s[s]) * f;
                double T = T_s[s] + (T_e[s] - T_s[s]) * f;
                for (int cy = 0; cy < NB; ++cy) {
                    int64_t b = (int64_t)nb * (iy - H) + cy;
                    double wy = sigma_T[s] > 0.0 ? cell_weight((double)b * bin, (double)(b + 1) * bin, v, sigma_T[s])
                                                 : ((int64_t)floor(v / bin) == b ? 1.0 : 0.0);
                    if (wy == 0.0) continue;
                    for (int cx = 0; cx < NB; ++cx) {
                        int64_t a = (int64_t)nb * (ix - H) + cx;
                        double wx = sigma_T[s] > 0.0 ? cell_weight((double)a * bin, (double)(a + 1) * bin, u, sigma_T[s])
                                                     : ((int64_t)floor(u / bin) == a ? 1.0 : 0.0);
                        if (wx == 0.0) continue;
                        for (int k = 0; k < K; ++k) {
                            int64_t j = (int64_t)nidx - k;
                            if (j < 0 || j > j_max) continue;
                            double t_lo = p->t_origin + (double)j * p->dt, t_hi = p->t_origin + (double)(j + 1) * p->dt;
                            double wt = sigma_t[s] > 0.0 ? cell_weight(t_lo, t_hi, T, sigma_t[s])
                                                         : ((int64_t)floor((T - p->t_origin) / p->dt) == j ? 1.0 : 0.0);
                            acc += (q_a[s] / (double)N) * wx * wy * wt * (double)lut[((size_t)cy * NB + cx) * K + k];
                        }
                    }
                }
            }
        }
        wave[nidx] = acc;
    }
}

/* ---------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon et al., SC'11), counter (c0..c3), key (k0,k1).  BASELINE north_star: noise is
 * keyed by (seed, pixel id, tick).  Reading D16: counter = (pixel_id, tick, 0, 0), key = (seed_lo, seed_hi).
 * ------------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1, n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* three standard normals for (pixel, tick): z_d, z_u from (u0,u1), z_r from (u2,u3) (Box-Muller),
 * u_i = (x_i + 0.5) 2^-32. */
void orc_noise_normals(uint64_t seed, uint32_t pixel_id, uint32_t tick, double z[3])
{
    uint32_t ctr[4] = { pixel_id, tick, 0u, 0u }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
    orc_philox4x32_10(ctr, key, x);
    const double two_pi = 6.283185307179586476925286766559;
    double u0 = ((double)x[0] + 0.5) * (1.0 / 4294967296.0), u1 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
    double u2 = ((double)x[2] + 0.5) * (1.0 / 4294967296.0), u3 = ((double)x[3] + 0.5) * (1.0 / 4294967296.0);
    double r01 = sqrt(-2.0 * log(u0)), r23 = sqrt(-2.0 * log(u2));
    z[0] = r01 * cos(two_pi * u1);
    z[1] = r01 * sin(two_pi * u1);
    z[2] = r23 * cos(two_pi * u3);
}

/* ---------------------------------------------------------------------------------------------
 * O6  LArPix-style electronics on ONE pixel; details D11-D17.
 *   per tick n: q += I_p[n]; ARMED and q >= threshold (+ discriminator noise) -> HOLD from n_c = n;
 *   at n == n_c + hold_ticks: q_s = q + uncorrelated noise; V = v_ped + gain*q_s/1000;
 *   adc = clamp(floor((V - v_cm)/(v_ref - v_cm) * 2^bits), 0, 2^bits - 1); hit (n, adc);
 *   q = reset noise; ARMED again from n+1, but not before min_spacing_ticks after the sample.
 *   Optional periodic reset of an ARMED channel every periodic_reset_ticks.
 *   Returns the number of hits (all of them counted, at most max_hits stored).
 * ------------------------------------------------------------------------------------------- */
int orc_electronics(const orc_params *p, uint64_t seed, int32_t pixel_id, const double *wave,
                    int max_hits, int32_t *hit_tick, int32_t *hit_adc)
{
    double q = 0.0;
    int armed = 1, n_c = 0, nhits = 0;
    int64_t rearm_at = 0;
    const double full = ldexp(1.0, p->adc_bits);
    for (int n = 0; n < p->n_ticks; ++n) {
        double z[3] = { 0.0, 0.0, 0.0 };
        int have_z = 0;
        if (p->noise_disc_e != 0.0) { orc_noise_normals(seed, (uint32_t)pixel_id, (uint32_t)n, z); have_z = 1; }
        if (armed && p->periodic_reset_ticks > 0 && n > 0 && (n % p->periodic_reset_ticks) == 0) q = 0.0;
        q += wave[n];                                                     /* CSA integrates */
        if (armed && n >= rearm_at && q >= p->threshold_e + p->noise_disc_e * z[0]) { armed = 0; n_c = n; }
        if (!armed && n == n_c + p->hold_ticks) {                         /* digitise 1.6 us after the crossing */
            if (!have_z && (p->noise_uncorr_e != 0.0 || p->noise_reset_e != 0.0))
                orc_noise_normals(seed, (uint32_t)pixel_id, (uint32_t)n, z);
            double q_s = q + p->noise_uncorr_e * z[1];
            double V = p->v_ped + p->gain_mv_per_ke * q_s / 1000.0;
            double a = floor((V - p->v_cm) / (p->v_ref - p->v_cm) * full);
            if (a < 0.0) a = 0.0;
            if (a > full - 1.0) a = full - 1.0;
            if (nhits < max_hits) { hit_tick[nhits] = n; hit_adc[nhits] = (int32_t)a; }
            ++nhits;
            q = p->noise_reset_e * z[2];                                  /* reset: collected charge discarded */
            armed = 1;
            /* next sample (crossing + hold) must come >= min_spacing_ticks after this one */
            rearm_at = (int64_t)n + 1;
            if ((int64_t)n + p->min_spacing_ticks - p->hold_ticks > rearm_at)
                rearm_at = (int64_t)n + p->min_spacing_ticks - p->hold_ticks;
        }
    }
    return nhits;
}

/* ---------------------------------------------------------------------------------------------
 * O7  Truth association: which segments fed a hit, and with what share of its charge.
 *   The paper describes truth propagation for the light path only (section 4.4: "the true track segment
 *   id ... contributing to each ADC sample"); this is the charge-side analogue, reading D26:
 *   - By eqs. (3.7)-(3.9) the current on a pixel is a sum over segments, I_p[n] = sum_s I_{p,s}[n], where I_{p,s} is
 *     eq. (3.9) evaluated for segment s alone (orc_pixel_current on a one-segment input).
 *   - At the sample tick n_h of hit h the CSA of O6 holds q = (reset noise) + sum_{n = n0}^{n_h} I_p[n], n0 = the first
 *     tick integrated since q was last set: the tick after the previous sample of that pixel (0 for its first hit),
 *     or a later periodic-reset tick r = k * periodic_reset_ticks (k >= 1) with r <= n_h - hold_ticks, the crossing tick
 *     (O6 clears q BEFORE it adds the charge of tick r, and only while armed, i.e. up to and including the crossing tick).
 *   - Share of segment s in hit h:  q_{h,s} = sum_{n = n0}^{n_h} I_{p,s}[n]  (electrons; signed, a bipolar induced
 *     current can make it negative); fraction f_{h,s} = q_{h,s} / sum_{s'} q_{h,s'}.  Noise belongs to no segment.
 * ------------------------------------------------------------------------------------------- */

/* I_{p,s} for the listed segments: waves[n_sel][n_ticks], one orc_pixel_current call per segment on that segment alone. */
void orc_segment_currents(const orc_params *p, const orc_tpc *tpcs, int tpc_index, const float *lut,
                          const int32_t *tpc, const double *q_a, const double *sigma_T, const double *sigma_t,
                          const double *u_s, const double *v_s, const double *u_e, const double *v_e,
                          const double *T_s, const double *T_e, const int32_t *n_samples,
                          int ix, int iy, int64_t n_sel, const int64_t *sel, double *waves)
{
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t k = 0; k < n_sel; ++k) {
        const int64_t s = sel[k];
        orc_pixel_current(p, tpcs, tpc_index, lut, 1, tpc + s, q_a + s, sigma_T + s, sigma_t + s,
                          u_s + s, v_s + s, u_e + s, v_e + s, T_s + s, T_e + s, n_samples + s,
                          ix, iy, waves + (size_t)k * p->n_ticks);
    }
}

/* hit_tick[n_hits]: the sample ticks of ONE pixel in increasing order (orc_electronics); seg_waves[n_sel][n_ticks].
 * Out: n0[n_hits] first integrated tick of each hit, share[n_hits][n_sel] = q_{h,s}. */
void orc_hit_truth(const orc_params *p, int n_hits, const int32_t *hit_tick,
                   int64_t n_sel, const double *seg_waves, int32_t *n0, double *share)
{
    for (int h = 0; h < n_hits; ++h) {
        int start = h > 0 ? hit_tick[h - 1] + 1 : 0;
        if (p->periodic_reset_ticks > 0) {
            int crossing = hit_tick[h] - p->hold_ticks;
            int r = (crossing / p->periodic_reset_ticks) * p->periodic_reset_ticks;   /* last reset tick <= crossing */
            if (r >= 1 && r > start) start = r;
        }
        n0[h] = start;
        for (int64_t k = 0; k < n_sel; ++k) {
            const double *w = seg_waves + (size_t)k * p->n_ticks;
            double q = 0.0;
            for (int n = start; n <= hit_tick[h]; ++n) q += w[n];
            share[(size_t)h * n_sel + k] = q;
        }
    }
}

/* =============================================================================================
 * Light simulation, eqs. (4.1)-(4.6); readings D28-D33 of DESIGN.md.
 * Test infrastructure like the rest of this file; shares nothing with the CUDA path.
 * ============================================================================================= */
typedef struct {
    double w_ph, w_ion;                 /* MeV per photon at zero field, MeV per electron */
    double dt, t_start;                 /* simulation tick delta_t and the time of tick 0, us */
    int    n_ticks;
    int    lut_m, n_lut_t;              /* LUT time bin = lut_m ticks (D29), LUT time bins */
    double vx0, vy0, vz0, vsize;        /* voxel grid origin and voxel edge, cm */
    int    nvx, nvy, nvz, n_det;
    double f_prompt, tau_p, tau_s;      /* eq. (4.4): ~0.3, ~0.007 us, ~1.6 us */
    double trunc_tau;                   /* convolution truncated at trunc_tau * tau_s (5) */
    double normal_above;                /* Poisson below, normal at or above this mean (30 p.e.) */
    int    n_resp;                      /* taps of the impulse response, sampled at delta_t (D32) */
    int    n_noise;                     /* sinusoids of the noise model (0 = no noise) */
} orc_light_params;

/* O8  Incident light, eqs. (4.1)(4.2).
 *   N_gamma,j = (1/W_ph - R_j/W_ion) dE_j = dE_j / W_ph - n_e,j   (n_e,j = R_j dE_j / W_ion of O1; clamped at >= 0)
 *   N_pe,ij   = eps_i V_i[voxel of segment j] N_gamma,j
 * Reading D28: the voxel is the one holding the segment's midpoint; a midpoint outside the voxel grid sees no light
 * (vox = -1); the deposition time t_0 of eq. (4.3) is the mean of the two end times, its tick k0 = floor((t_0 - t_start)/dt).
 * npe is [n_det][n] (sensor-major). */
void orc_light_npe(const orc_light_params *p, int64_t n,
                   const float *xs, const float *ys, const float *zs, const float *ts,
                   const float *xe, const float *ye, const float *ze, const float *te, const float *dE,
                   const double *n_e, const float *eff, const float *vis,
                   int32_t *vox, int32_t *k0, double *n_gamma, double *npe)
{
    const int64_t nvox = (int64_t)p->nvx * p->nvy * p->nvz;
    for (int64_t j = 0; j < n; ++j) {
        double xm = 0.5 * ((double)xs[j] + (double)xe[j]), ym = 0.5 * ((double)ys[j] + (double)ye[j]);
        double zm = 0.5 * ((double)zs[j] + (double)ze[j]), t0 = 0.5 * ((double)ts[j] + (double)te[j]);
        double ng = (double)dE[j] / p->w_ph - n_e[j];
        if (!(ng > 0.0)) ng = 0.0;
        n_gamma[j] = ng;
        k0[j] = (int32_t)floor((t0 - p->t_start) / p->dt);
        int64_t ix = (int64_t)floor((xm - p->vx0) / p->vsize), iy = (int64_t)floor((ym - p->vy0) / p->vsize);
        int64_t iz = (int64_t)floor((zm - p->vz0) / p->vsize);
        int inside = ix >= 0 && ix < p->nvx && iy >= 0 && iy < p->nvy && iz >= 0 && iz < p->nvz;
        vox[j] = inside ? (int32_t)((iz * p->nvy + iy) * p->nvx + ix) : -1;
        for (int i = 0; i < p->n_det; ++i)
            npe[(size_t)i * n + j] = inside ? (double)eff[i] * (double)vis[(size_t)i * nvox + vox[j]] * ng : 0.0;
    }
}

/* O9  Photocurrent time profile, eq. (4.3).  Reading D29: f_i[voxel][b] is the fraction of the sensor's light
 * that arrives during LUT time bin b (it sums to 1 over b), a LUT bin spans lut_m simulation ticks, and I_pe is kept in
 * photoelectrons PER TICK: segment j adds N_pe,ij f_i[vox_j][b] / lut_m to each of the ticks k0_j + b lut_m + r, r = 0 ..
 * lut_m - 1, inside [0, n_ticks).  (The printed prefactor Delta_t_LUT / delta_t and the printed sum index are garbled,
 * SURVEY D20; this is the reading that conserves photoelectrons.)  ipe is [n_det][n_ticks], overwritten. */
void orc_light_profile(const orc_light_params *p, int64_t n, const int32_t *vox, const int32_t *k0,
                       const double *npe, const float *tprof, double *ipe)
{
    const int64_t nvox = (int64_t)p->nvx * p->nvy * p->nvz;
    memset(ipe, 0, sizeof(double) * (size_t)p->n_det * p->n_ticks);
    for (int i = 0; i < p->n_det; ++i)
        for (int64_t j = 0; j < n; ++j) {
            if (vox[j] < 0) continue;
            const float *f = tprof + ((size_t)i * nvox + vox[j]) * p->n_lut_t;
            for (int b = 0; b < p->n_lut_t; ++b)
                for (int r = 0; r < p->lut_m; ++r) {
                    int64_t t = (int64_t)k0[j] + (int64_t)b * p->lut_m + r;
                    if (t >= 0 && t < p->n_ticks) ipe[(size_t)i * p->n_ticks + t] += npe[(size_t)i * n + j] * (double)f[b] / (double)p->lut_m;
                }
        }
}

/* O10  Scintillation time structure, eqs. (4.4)(4.5).
 *   f_scint(t) = f_p/tau_p exp(-t/tau_p) + (1 - f_p)/tau_s exp(-t/tau_s)
 *   I_scint[t] = sum_{s = 0}^{s_max} I_pe[t - s] w[s],   s_max = floor(trunc_tau tau_s / dt)
 * Reading D30: eq. (4.5) multiplies a per-tick quantity by the density f_scint((i_t - j_t) dt); the weight of lag s is taken
 * as the integral of f_scint over that tick,
 *   w[s] = f_p (e^{-s dt/tau_p} - e^{-(s+1) dt/tau_p}) + (1 - f_p) (e^{-s dt/tau_s} - e^{-(s+1) dt/tau_s}),
 * which is f_scint(s dt) dt to first order in dt/tau and conserves the light for any tick (point samples of the 7 ns
 * component at a 16 ns tick would add up to 1.46).  w[s_max + 1] receives the weights; isc is [n_det][n_ticks]. */
int orc_light_scint_weights(const orc_light_params *p, double *w, int cap)
{
    const int s_max = (int)floor(p->trunc_tau * p->tau_s / p->dt);
    for (int s = 0; s <= s_max && s < cap; ++s) {
        double t = (double)s * p->dt;
        w[s] = p->f_prompt * (exp(-t / p->tau_p) - exp(-(t + p->dt) / p->tau_p)) +
               (1.0 - p->f_prompt) * (exp(-t / p->tau_s) - exp(-(t + p->dt) / p->tau_s));
    }
    return s_max;
}

/* truncated causal convolution out[i][t] = scale_i sum_{s=0}^{n_w-1} in[i][t-s] w[s]: eq. (4.5) with scale 1, and the sum
 * of eq. (4.6) with scale G_i */
void orc_light_convolve(int n_det, int n_ticks, const double *in, const double *w, int n_w, const float *scale, double *out)
{
#pragma omp parallel for schedule(static)
    for (int i = 0; i < n_det; ++i)
        for (int t = 0; t < n_ticks; ++t) {
            double acc = 0.0;
            for (int s = 0; s < n_w && s <= t; ++s) acc += in[(size_t)i * n_ticks + t - s] * w[s];
            out[(size_t)i * n_ticks + t] = (scale ? (double)scale[i] : 1.0) * acc;
        }
}

/* O11  Counting statistics per time profile bin: inverse-transform-sampling Poisson below `normal_above`
 * expected photoelectrons (30), N(lambda, sqrt(lambda)) at or above.  Reading D31: the uniforms of (sensor i, tick t) are
 * u_k = (x_k + 0.5) 2^-32 of Philox4x32-10(counter (i, t, 0, 0x4C474854 'LGHT'), key = seed); Poisson: the smallest k with
 * CDF(k) >= u_0 (k = 0, p = exp(-lambda), c = p; while u_0 > c: k += 1, p *= lambda / k, c += p; at most 200 steps);
 * normal: lambda + sqrt(lambda) sqrt(-2 ln u_0) cos(2 pi u_1), not rounded, not clamped.  lambda <= 0 gives 0. */
double orc_light_fluctuate_one(const orc_light_params *p, uint64_t seed, uint32_t det, uint32_t tick, double lambda)
{
    if (!(lambda > 0.0)) return 0.0;
    uint32_t ctr[4] = { det, tick, 0u, 0x4C474854u }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
    orc_philox4x32_10(ctr, key, x);
    const double u0 = ((double)x[0] + 0.5) * (1.0 / 4294967296.0), u1 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
    if (lambda < p->normal_above) {
        int k = 0;
        double pk = exp(-lambda), c = pk;
        while (u0 > c && k < 200) { ++k; pk *= lambda / (double)k; c += pk; }
        return (double)k;
    }
    return lambda + sqrt(lambda) * (sqrt(-2.0 * log(u0)) * cos(6.283185307179586476925286766559 * u1));
}

void orc_light_fluctuate(const orc_light_params *p, uint64_t seed, const double *isc, double *nobs)
{
    for (int i = 0; i < p->n_det; ++i)
        for (int t = 0; t < p->n_ticks; ++t)
            nobs[(size_t)i * p->n_ticks + t] = orc_light_fluctuate_one(p, seed, (uint32_t)i, (uint32_t)t, isc[(size_t)i * p->n_ticks + t]);
}

/* O12  Light read-out electronics, eq. (4.6): V_i[t] = n_i[t] + G_i sum_s N_obs,i[t - s] i_resp[s]
 * (reading D32: the response model is sampled at the simulation tick, Delta_t_resp / delta_t = 1; it is unit-normalised
 * by its provider).  Noise (reading D33): "random phase sinusoids with appropriate amplitudes" from a user-given spectrum:
 * n_i[t] = sum_f A_f cos(2 pi k_f t / n_ticks + phi_if), phi_if = 2 pi u_0 of Philox(counter (i, f, 1, 'LGHT'), key = seed). */
void orc_light_noise(const orc_light_params *p, uint64_t seed, const float *amp, const int32_t *kf, double *noise)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int i = 0; i < p->n_det; ++i) {
        for (int t = 0; t < p->n_ticks; ++t) noise[(size_t)i * p->n_ticks + t] = 0.0;
        for (int f = 0; f < p->n_noise; ++f) {
            uint32_t ctr[4] = { (uint32_t)i, (uint32_t)f, 1u, 0x4C474854u }, key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) }, x[4];
            orc_philox4x32_10(ctr, key, x);
            const double phi = two_pi * (((double)x[0] + 0.5) * (1.0 / 4294967296.0));
            for (int t = 0; t < p->n_ticks; ++t)
                noise[(size_t)i * p->n_ticks + t] += (double)amp[f] * cos(two_pi * (double)kf[f] * (double)t / (double)p->n_ticks + phi);
        }
    }
}
