// Light simulation: eqs. (4.1)-(4.6) of arXiv 2212.09807; readings D28-D33.
//
//   L1 light_npe_kernel       thread = segment: photon yield, voxel and deposition tick (float64 index path, as S2 / S3),
//                             N_pe for every sensor (the visibility LUT is a gather), tick histogram for the sort
//   L2 light_tick_sum_kernel  segments counting-sorted by deposition tick (lists sorted by segment id, so every sum below has a
//      light_profile_kernel   fixed order); CTA = (sensor, deposition tick): the light of that tick's segments per LUT time bin;
//                             thread = (sensor, tick): adds the LUT bins of the deposition ticks that reach it
//   L3 / L5 light_conv_kernel truncated causal convolution, CTA = (sensor, 256 ticks): input window and weights in shared
//                             memory, ascending lag; L5 also scales by the gain and adds the noise sinusoids
//   L4 light_fluct_kernel     thread = (sensor, tick): Philox4x32-10, inverse-transform Poisson / Box-Muller normal in float64
// The paper gives each of these a plain 2-D grid with a loop over ALL segments per (sensor, tick); here the tick
// sort cuts that loop to the segments inside the LUT's time span.  None of it is a dense contraction worth a tensor core at
// the sizes of P:L778 (a 501-tap convolution of n_det x n_ticks samples is ~1e9 multiply-adds): FP32 pipe, shared memory.
#include <math.h>
#include <algorithm>
#include <vector>
#include "common.cuh"
#include "scan.cuh"

struct LightDev {
    double w_ph, dt, t_start, vx0, vy0, vz0, vsize, normal_above;
    int n_ticks, lut_m, n_lut_t, nvx, nvy, nvz, n_det, n_resp, n_noise, n_scint, span;   // span = n_lut_t * lut_m ticks
    long long nvox;
};

struct lartpc_light {
    lartpc_light_params_t params;
    LightDev d;
    int device = 0;
    float *eff = nullptr, *gain = nullptr, *vis = nullptr, *tprof = nullptr, *resp = nullptr, *w_scint = nullptr;
    float *noise_amp = nullptr, *phase = nullptr;   int32_t *noise_k = nullptr;
    // tick sort scratch: keys k0 + span - 1 in [0, n_keys)
    int n_keys = 0;
    int32_t *key_count = nullptr, *key_offs = nullptr, *key_start = nullptr;   int64_t table_cap = 0;   // [n_keys][blocks] (+1)
    int32_t *list = nullptr;  int64_t list_cap = 0;
    float *tick_sums = nullptr;                    // A[n_det][n_keys][n_lut_t] of light_tick_sum_kernel
    long long *scan_tmp = nullptr;
};

namespace {

constexpr unsigned LGHT = 0x4C474854u;

__global__ void __launch_bounds__(256)
light_npe_kernel(LightDev d, SegPtrs s, int64_t n, const float *__restrict__ n_e, const float *__restrict__ eff,
                 const float *__restrict__ vis, int32_t *vox, int32_t *k0, float *n_gamma, float *npe, int32_t *key_count)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    // float64, individually rounded, in the oracle's order: the voxel and the tick are integer decisions
    const double xm = xmul(0.5, xadd((double)s.xs[j], (double)s.xe[j])), ym = xmul(0.5, xadd((double)s.ys[j], (double)s.ye[j]));
    const double zm = xmul(0.5, xadd((double)s.zs[j], (double)s.ze[j])), t0 = xmul(0.5, xadd((double)s.ts[j], (double)s.te[j]));
    double ng = xsub(xdiv((double)s.dE[j], d.w_ph), (double)n_e[j]);           // eq. (4.1) over the segment: dE / W_ph - n_e
    if (!(ng > 0.0)) ng = 0.0;
    const int k = (int)floor(xdiv(xsub(t0, d.t_start), d.dt));
    const long long ix = (long long)floor(xdiv(xsub(xm, d.vx0), d.vsize)), iy = (long long)floor(xdiv(xsub(ym, d.vy0), d.vsize));
    const long long iz = (long long)floor(xdiv(xsub(zm, d.vz0), d.vsize));
    const bool inside = ix >= 0 && ix < d.nvx && iy >= 0 && iy < d.nvy && iz >= 0 && iz < d.nvz;
    const int v = inside ? (int)((iz * d.nvy + iy) * d.nvx + ix) : -1;
    vox[j] = v;
    k0[j] = k;
    n_gamma[j] = (float)ng;
    const float ngf = (float)ng;
    for (int i = 0; i < d.n_det; ++i)                                           // eq. (4.2)
        npe[(size_t)i * n + j] = inside ? eff[i] * __ldg(vis + (size_t)i * d.nvox + v) * ngf : 0.f;
    (void)key_count;
}

// Stable counting sort of the segments by deposition tick (key = k0 + span - 1 in [0, n_keys); a segment without light or
// whose light misses the waveform has no key): count per (key, block of SORT_B segments), exclusive scan over the
// [key][block] table, then every segment goes to offset[key][block] + its rank among the earlier segments of its block with
// the same key.  No order-dependent atomics: the list of a tick is in segment order, run after run.
constexpr int SORT_T = 256, SORT_B = 2048;
__device__ __forceinline__ int light_key(const LightDev &d, int n_keys, int vox, int k0)
{
    const long long key = (long long)k0 + d.span - 1;
    return (vox >= 0 && key >= 0 && key < n_keys) ? (int)key : -1;
}

__global__ void __launch_bounds__(SORT_T)
light_key_count_kernel(LightDev d, int n_keys, int64_t n, int n_blocks, const int32_t *__restrict__ vox,
                       const int32_t *__restrict__ k0, int32_t *count)
{
    for (int q = threadIdx.x; q < SORT_B; q += SORT_T) {
        const int64_t j = (int64_t)blockIdx.x * SORT_B + q;
        if (j >= n) break;
        const int key = light_key(d, n_keys, vox[j], k0[j]);
        if (key >= 0) atomicAdd(&count[(size_t)key * n_blocks + blockIdx.x], 1);   // a counter: the order of the adds is immaterial
    }
}

__global__ void light_key_start_kernel(int n_keys, int n_blocks, const int32_t *__restrict__ offs, int32_t *key_start)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k <= n_keys) key_start[k] = offs[(size_t)k * n_blocks];                  // offs[n_keys * n_blocks] = total
}

__global__ void __launch_bounds__(SORT_T)
light_key_scatter_kernel(LightDev d, int n_keys, int64_t n, int n_blocks, const int32_t *__restrict__ vox,
                         const int32_t *__restrict__ k0, const int32_t *__restrict__ offs, int32_t *list)
{
    __shared__ int s_key[SORT_B];
    const int64_t base = (int64_t)blockIdx.x * SORT_B;
    for (int q = threadIdx.x; q < SORT_B; q += SORT_T)
        s_key[q] = base + q < n ? light_key(d, n_keys, vox[base + q], k0[base + q]) : -1;
    __syncthreads();
    for (int q = threadIdx.x; q < SORT_B; q += SORT_T) {
        const int key = s_key[q];
        if (key < 0) continue;
        int rank = 0;
        for (int r = 0; r < q; ++r) rank += s_key[r] == key;
        list[offs[(size_t)key * n_blocks + blockIdx.x] + rank] = (int32_t)(base + q);
    }
}

struct CountF { const int32_t *v; __device__ long long operator()(int64_t i) const { return v[i]; } };

// Eq. (4.3) in two steps.  (1) CTA = (deposition tick k, sensor i): A[i][k][b] = sum over the segments of that tick of
// N_pe,ij f_i[vox_j][b], all LUT time bins b at once (the profile of a voxel is one contiguous read).  A spill puts the 1e4
// segments of an interaction into ONE tick, so the list is cut into contiguous chunks, one per group of P lanes (P = LUT
// bins rounded up to a power of two; 256 threads = 256 / P groups), each summed in list order with compensated (Kahan)
// float32 additions, the chunks then added in chunk order: a fixed order whatever the launch.  (2) thread = (sensor, tick
// t): ipe[i][t] = sum over k0 in [t - span + 1, t] of A[i][k0][(t - k0) / lut_m] / lut_m.
constexpr int TS_THREADS = 256;
__global__ void __launch_bounds__(TS_THREADS)
light_tick_sum_kernel(LightDev d, int64_t n, int P, const int32_t *__restrict__ vox, const float *__restrict__ npe,
                      const float *__restrict__ tprof, const int32_t *__restrict__ key_start, const int32_t *__restrict__ list,
                      float *A)
{
    __shared__ float s_part[TS_THREADS];
    const int key = blockIdx.x, i = blockIdx.y, tid = threadIdx.x;
    const int e0 = key_start[key], len = key_start[key + 1] - e0;
    float *out = A + ((size_t)i * gridDim.x + key) * d.n_lut_t;
    if (len == 0) {                                                             // CTA-uniform
        if (tid < d.n_lut_t) out[tid] = 0.f;
        return;
    }
    const int b = tid & (P - 1), g = tid / P, n_groups = TS_THREADS / P;
    const int chunk = (len + n_groups - 1) / n_groups;
    const int c0 = min(g * chunk, len), c1 = min(c0 + chunk, len);
    const float *np_i = npe + (size_t)i * n;
    const float *tp_i = tprof + (size_t)i * d.nvox * d.n_lut_t;
    float acc = 0.f, comp = 0.f;
    if (b < d.n_lut_t) {
#pragma unroll 4
        for (int e = e0 + c0; e < e0 + c1; ++e) {
            const int j = __ldg(list + e);
            const float y = __fmul_rn(__ldg(np_i + j), __ldg(tp_i + (size_t)__ldg(vox + j) * d.n_lut_t + b)) - comp;
            const float sum = __fadd_rn(acc, y);
            comp = __fsub_rn(__fsub_rn(sum, acc), y);
            acc = sum;
        }
    }
    s_part[tid] = acc;
    __syncthreads();
    if (tid < d.n_lut_t) {
        float tot = 0.f;
        for (int q = 0; q < n_groups; ++q) tot += s_part[q * P + tid];
        out[tid] = tot;
    }
}

__global__ void __launch_bounds__(128)
light_profile_kernel(LightDev d, int n_keys, const float *__restrict__ A, float *ipe)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (t >= d.n_ticks) return;
    const float *Ai = A + (size_t)i * n_keys * d.n_lut_t;
    float acc = 0.f;
    for (int key = t; key < t + d.span; ++key)                                  // key = k0 + span - 1
        acc += Ai[(size_t)key * d.n_lut_t + (t + d.span - 1 - key) / d.lut_m];
    ipe[(size_t)i * d.n_ticks + t] = acc / (float)d.lut_m;                      // photoelectrons per tick (D29)
}

// out[i][t] = scale_i * sum_{s=0}^{min(n_w-1, t)} in[i][t-s] w[s]  (+ noise).  CTA = (256 ticks, sensor); the input window
// [t_lo - (n_w - 1), t_lo + 255] and the weights sit in shared memory; ascending lag as the oracle.
constexpr int CONV_T = 256;
__global__ void __launch_bounds__(CONV_T)
light_conv_kernel(int n_det, int n_ticks, const float *__restrict__ in, const float *__restrict__ w, int n_w,
                  const float *__restrict__ scale, int n_noise, const float *__restrict__ noise_amp,
                  const int32_t *__restrict__ noise_k, const float *__restrict__ phase, float *out)
{
    extern __shared__ float sm[];
    float *s_w = sm, *s_in = sm + n_w;                                          // [n_w], [n_w - 1 + CONV_T]
    const int i = blockIdx.y, t_lo = blockIdx.x * CONV_T, tid = threadIdx.x;
    const float *x = in + (size_t)i * n_ticks;
    for (int k = tid; k < n_w; k += CONV_T) s_w[k] = w[k];
    for (int k = tid; k < n_w - 1 + CONV_T; k += CONV_T) {
        const int t = t_lo - (n_w - 1) + k;
        s_in[k] = (t >= 0 && t < n_ticks) ? x[t] : 0.f;
    }
    __syncthreads();
    const int t = t_lo + tid;
    if (t >= n_ticks) return;
    const float *xi = s_in + (n_w - 1) + tid;                                   // xi[-s] = in[t - s] (0 before the waveform)
    float acc = 0.f;
    for (int s = 0; s < n_w; ++s) acc = fmaf(xi[-s], s_w[s], acc);
    float v = (scale ? scale[i] : 1.f) * acc;
    if (n_noise > 0) {
        // n_i[t] = sum_f A_f cos(2 pi k_f t / n_ticks + phi_if) (D33); the argument is reduced in integers first
        float nz = 0.f;
        for (int f = 0; f < n_noise; ++f) {
            const int r = (int)(((long long)noise_k[f] * t) % n_ticks);
            nz += noise_amp[f] * cosf(6.283185307f * ((float)r / (float)n_ticks) + phase[i * n_noise + f]);
        }
        v += nz;
    }
    out[(size_t)i * n_ticks + t] = v;
}

__global__ void light_phase_kernel(int n_det, int n_noise, unsigned long long seed, float *phase)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n_det * n_noise) return;
    uint32_t x[4];
    philox4x32_10((uint32_t)(q / n_noise), (uint32_t)(q % n_noise), 1u, LGHT, (uint32_t)seed, (uint32_t)(seed >> 32), x);
    phase[q] = (float)(6.283185307179586476925286766559 * (((double)x[0] + 0.5) * (1.0 / 4294967296.0)));
}

// P:L782 / D31: float64 decisions on the float32 mean
__global__ void __launch_bounds__(256)
light_fluct_kernel(LightDev d, unsigned long long seed, const float *__restrict__ isc, float *nobs)
{
    const int64_t q = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (int64_t)d.n_det * d.n_ticks) return;
    const double lambda = (double)isc[q];
    float r = 0.f;
    if (lambda > 0.0) {
        uint32_t x[4];
        philox4x32_10((uint32_t)(q / d.n_ticks), (uint32_t)(q % d.n_ticks), 0u, LGHT, (uint32_t)seed, (uint32_t)(seed >> 32), x);
        const double u0 = ((double)x[0] + 0.5) * (1.0 / 4294967296.0), u1 = ((double)x[1] + 0.5) * (1.0 / 4294967296.0);
        if (lambda < d.normal_above) {
            int k = 0;
            double pk = exp(-lambda), c = pk;
            while (u0 > c && k < 200) { ++k;  pk = xmul(pk, xdiv(lambda, (double)k));  c = xadd(c, pk); }
            r = (float)k;
        } else {
            r = (float)(lambda + sqrt(lambda) * (sqrt(-2.0 * log(u0)) * cos(6.283185307179586476925286766559 * u1)));
        }
    }
    nobs[q] = r;
}

}  // namespace

// ---- host side ------------------------------------------------------------------------------------------------------
static void light_free(lartpc_light *l)
{
    if (!l) return;
    cudaFree(l->eff); cudaFree(l->gain); cudaFree(l->vis); cudaFree(l->tprof); cudaFree(l->resp); cudaFree(l->w_scint);
    cudaFree(l->noise_amp); cudaFree(l->phase); cudaFree(l->noise_k);
    cudaFree(l->key_count); cudaFree(l->key_start); cudaFree(l->key_offs); cudaFree(l->list); cudaFree(l->scan_tmp); cudaFree(l->tick_sums);
    delete l;
}

template <typename T> static cudaError_t upload(T **dst, const T *src, size_t n)
{
    cudaError_t e = cudaMalloc(dst, sizeof(T) * (n ? n : 1));
    if (e == cudaSuccess && n) e = cudaMemcpy(*dst, src, sizeof(T) * n, cudaMemcpyHostToDevice);
    return e;
}

extern "C" int lartpc_light_create(const lartpc_light_params_t *p, const float *eff, const float *gain, const float *vis,
                                   const float *tprof, const float *resp, const float *noise_amp, const int32_t *noise_k,
                                   lartpc_light_t **out)
{
    if (!p || !eff || !gain || !vis || !tprof || !resp || !out) return LARTPC_ERR_BAD_ARGUMENT;
    if (p->n_ticks < 1 || p->lut_m < 1 || p->n_lut_t < 1 || p->nvx < 1 || p->nvy < 1 || p->nvz < 1 || p->n_det < 1 ||
        p->n_resp < 1 || p->n_noise < 0 || !(p->tick_us > 0.0) || !(p->vox_size_cm > 0.0) || !(p->w_ph_mev > 0.0) ||
        !(p->tau_prompt_us > 0.0) || !(p->tau_slow_us > 0.0) || !(p->trunc_tau > 0.0) || (p->n_noise > 0 && (!noise_amp || !noise_k)))
        return LARTPC_ERR_BAD_ARGUMENT;
    if ((long long)p->n_ticks * p->n_det >= (1ll << 31) || (long long)p->nvx * p->nvy * p->nvz >= (1ll << 31)) return LARTPC_ERR_UNSUPPORTED;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return LARTPC_ERR_CUDA;
    if (prop.major != 10) return LARTPC_ERR_DEVICE;
    lartpc_light *l = new lartpc_light();
    l->params = *p;
    l->device = dev;
    LightDev &d = l->d;
    d.w_ph = p->w_ph_mev;  d.dt = p->tick_us;  d.t_start = p->t_start_us;
    d.vx0 = p->vox_x0;  d.vy0 = p->vox_y0;  d.vz0 = p->vox_z0;  d.vsize = p->vox_size_cm;  d.normal_above = p->normal_above;
    d.n_ticks = p->n_ticks;  d.lut_m = p->lut_m;  d.n_lut_t = p->n_lut_t;  d.nvx = p->nvx;  d.nvy = p->nvy;  d.nvz = p->nvz;
    d.n_det = p->n_det;  d.n_resp = p->n_resp;  d.n_noise = p->n_noise;  d.span = p->n_lut_t * p->lut_m;
    d.nvox = (long long)p->nvx * p->nvy * p->nvz;
    // eq. (4.4) integrated over a tick (D30), s = 0 .. floor(trunc_tau tau_s / dt), in float64 then rounded once
    const int s_max = (int)floor(p->trunc_tau * p->tau_slow_us / p->tick_us);
    d.n_scint = s_max + 1;
    std::vector<float> w((size_t)d.n_scint);
    for (int s = 0; s <= s_max; ++s) {
        const double t = (double)s * p->tick_us;
        w[s] = (float)(p->f_prompt * (exp(-t / p->tau_prompt_us) - exp(-(t + p->tick_us) / p->tau_prompt_us)) +
                       (1.0 - p->f_prompt) * (exp(-t / p->tau_slow_us) - exp(-(t + p->tick_us) / p->tau_slow_us)));
    }
    const size_t nvox = (size_t)d.nvox;
    l->n_keys = d.n_ticks + d.span - 1;
    cudaError_t e = upload(&l->eff, eff, (size_t)d.n_det);
    if (e == cudaSuccess) e = upload(&l->gain, gain, (size_t)d.n_det);
    if (e == cudaSuccess) e = upload(&l->vis, vis, (size_t)d.n_det * nvox);
    if (e == cudaSuccess) e = upload(&l->tprof, tprof, (size_t)d.n_det * nvox * d.n_lut_t);
    if (e == cudaSuccess) e = upload(&l->resp, resp, (size_t)d.n_resp);
    if (e == cudaSuccess) e = upload(&l->w_scint, w.data(), w.size());
    if (e == cudaSuccess) e = upload(&l->noise_amp, noise_amp, (size_t)d.n_noise);
    if (e == cudaSuccess) e = upload(&l->noise_k, noise_k, (size_t)d.n_noise);
    if (e == cudaSuccess) e = cudaMalloc(&l->phase, sizeof(float) * (size_t)(d.n_det * d.n_noise + 1));
    if (e == cudaSuccess) e = cudaMalloc(&l->key_start, sizeof(int32_t) * (size_t)(l->n_keys + 1));
    if (e == cudaSuccess) e = cudaMalloc(&l->tick_sums, sizeof(float) * (size_t)d.n_det * (size_t)l->n_keys * (size_t)d.n_lut_t);
    if (e != cudaSuccess) { lartpc_note_cuda_error(e, __FILE__, __LINE__);  light_free(l);  return LARTPC_ERR_CUDA; }
    *out = l;
    return LARTPC_OK;
}

extern "C" void lartpc_light_destroy(lartpc_light_t *l)
{
    if (!l) return;
    DeviceGuard dg(l->device);
    light_free(l);
}

extern "C" int lartpc_light_npe(lartpc_light_t *l, const lartpc_segments_t *seg, int64_t n, const float *n_e, int32_t *vox,
                                int32_t *k0, float *n_gamma, float *npe, void *stream)
{
    if (!l || !seg || n < 0 || (n > 0 && (!n_e || !vox || !k0 || !n_gamma || !npe))) return LARTPC_ERR_BAD_ARGUMENT;
    if (n == 0) return LARTPC_OK;
    if (n >= (1ll << 31)) return LARTPC_ERR_UNSUPPORTED;
    DeviceGuard dg(l->device);
    SegPtrs s{seg->xs, seg->ys, seg->zs, seg->ts, seg->xe, seg->ye, seg->ze, seg->te, seg->dE};
    ++g_lartpc_launches;
    light_npe_kernel<<<div_up(n, 256), 256, 0, (cudaStream_t)stream>>>(l->d, s, n, n_e, l->eff, l->vis, vox, k0, n_gamma, npe,
                                                                      nullptr);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

extern "C" int lartpc_light_profile(lartpc_light_t *l, int64_t n, const int32_t *vox, const int32_t *k0, const float *npe,
                                    float *ipe, void *stream)
{
    if (!l || n < 0 || !ipe || (n > 0 && (!vox || !k0 || !npe))) return LARTPC_ERR_BAD_ARGUMENT;
    if (n >= (1ll << 31)) return LARTPC_ERR_UNSUPPORTED;
    DeviceGuard dg(l->device);
    cudaStream_t st = (cudaStream_t)stream;
    const LightDev &d = l->d;
    if (n > l->list_cap) {
        if (l->list) cudaFree(l->list);
        l->list = nullptr;  l->list_cap = 0;
        LARTPC_CUDA_TRY(cudaMalloc(&l->list, sizeof(int32_t) * (size_t)(n + n / 8 + 1024)));
        l->list_cap = n + n / 8 + 1024;
    }
    // stable counting sort of the segments by deposition tick
    const int n_blocks = (int)std::max<int64_t>((n + SORT_B - 1) / SORT_B, 1);
    const int64_t table = (int64_t)l->n_keys * n_blocks;
    if (table + 1 >= (1ll << 31)) return LARTPC_ERR_UNSUPPORTED;
    if (table + 1 > l->table_cap) {
        cudaFree(l->key_count);  cudaFree(l->key_offs);  cudaFree(l->scan_tmp);
        l->key_count = l->key_offs = nullptr;  l->scan_tmp = nullptr;  l->table_cap = 0;
        LARTPC_CUDA_TRY(cudaMalloc(&l->key_count, sizeof(int32_t) * (size_t)(table + 1)));
        LARTPC_CUDA_TRY(cudaMalloc(&l->key_offs, sizeof(int32_t) * (size_t)(table + 1)));
        LARTPC_CUDA_TRY(cudaMalloc(&l->scan_tmp, sizeof(long long) * (size_t)lscan::tmp_elems(table + 1)));
        l->table_cap = table + 1;
    }
    LARTPC_CUDA_TRY(cudaMemsetAsync(l->key_count, 0, sizeof(int32_t) * (size_t)(table + 1), st));
    if (n > 0) {
        ++g_lartpc_launches;
        light_key_count_kernel<<<n_blocks, SORT_T, 0, st>>>(d, l->n_keys, n, n_blocks, vox, k0, l->key_count);
    }
    LARTPC_CUDA_TRY(lscan::exclusive_scan(table, CountF{l->key_count}, l->key_offs, true, (long long *)nullptr, l->scan_tmp, st));
    ++g_lartpc_launches;
    light_key_start_kernel<<<div_up(l->n_keys + 1, 256), 256, 0, st>>>(l->n_keys, n_blocks, l->key_offs, l->key_start);
    if (n > 0) {
        ++g_lartpc_launches;
        light_key_scatter_kernel<<<n_blocks, SORT_T, 0, st>>>(d, l->n_keys, n, n_blocks, vox, k0, l->key_offs, l->list);
    }
    int P = 1;
    while (P < d.n_lut_t) P <<= 1;
    if (P > TS_THREADS) return LARTPC_ERR_UNSUPPORTED;
    g_lartpc_launches += 2;
    light_tick_sum_kernel<<<dim3((unsigned)l->n_keys, (unsigned)d.n_det), TS_THREADS, 0, st>>>(
        d, n, P, vox, npe, l->tprof, l->key_start, l->list, l->tick_sums);
    light_profile_kernel<<<dim3((unsigned)div_up(d.n_ticks, 128), (unsigned)d.n_det), 128, 0, st>>>(d, l->n_keys, l->tick_sums, ipe);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

static int light_conv(lartpc_light *l, const float *in, const float *w, int n_w, const float *scale, int n_noise, float *out,
                      cudaStream_t st)
{
    const LightDev &d = l->d;
    const size_t smem = sizeof(float) * (size_t)(2 * n_w - 1 + CONV_T);
    if (smem > 200 * 1024) return LARTPC_ERR_UNSUPPORTED;             // (a 1 ns tick with tau_s = 1.6 us needs 65 KB)
    static SmemCfg cfg;
    LARTPC_CUDA_TRY(ensure_dyn_smem(light_conv_kernel, cfg, l->device, smem));
    ++g_lartpc_launches;
    light_conv_kernel<<<dim3((unsigned)div_up(d.n_ticks, CONV_T), (unsigned)d.n_det), CONV_T, smem, st>>>(
        d.n_det, d.n_ticks, in, w, n_w, scale, n_noise, l->noise_amp, l->noise_k, l->phase, out);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

extern "C" int lartpc_light_scintillation(lartpc_light_t *l, const float *ipe, float *isc, void *stream)
{
    if (!l || !ipe || !isc) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(l->device);
    return light_conv(l, ipe, l->w_scint, l->d.n_scint, nullptr, 0, isc, (cudaStream_t)stream);
}

extern "C" int lartpc_light_fluctuate(lartpc_light_t *l, uint64_t seed, const float *isc, float *nobs, void *stream)
{
    if (!l || !isc || !nobs) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(l->device);
    const int64_t q = (int64_t)l->d.n_det * l->d.n_ticks;
    ++g_lartpc_launches;
    light_fluct_kernel<<<div_up(q, 256), 256, 0, (cudaStream_t)stream>>>(l->d, seed, isc, nobs);
    LARTPC_CUDA_TRY(cudaGetLastError());
    return LARTPC_OK;
}

extern "C" int lartpc_light_electronics(lartpc_light_t *l, uint64_t seed, const float *nobs, float *v, void *stream)
{
    if (!l || !nobs || !v) return LARTPC_ERR_BAD_ARGUMENT;
    DeviceGuard dg(l->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (l->d.n_noise > 0) {
        ++g_lartpc_launches;
        light_phase_kernel<<<div_up((int64_t)l->d.n_det * l->d.n_noise, 128), 128, 0, st>>>(l->d.n_det, l->d.n_noise, seed, l->phase);
    }
    return light_conv(l, nobs, l->resp, l->d.n_resp, l->gain, l->d.n_noise, v, st);
}

static size_t al256(size_t x) { return (x + 255) & ~(size_t)255; }

extern "C" size_t lartpc_light_workspace_bytes(const lartpc_light_t *l, int64_t n)
{
    if (!l || n < 0) return 0;
    const size_t wf = al256(sizeof(float) * (size_t)l->d.n_det * l->d.n_ticks), sn = al256(sizeof(float) * (size_t)(n ? n : 1));
    return 3 * sn + al256(sizeof(float) * (size_t)l->d.n_det * (size_t)(n ? n : 1)) + 3 * wf + 256;
}

extern "C" int lartpc_light_run(lartpc_light_t *l, const lartpc_segments_t *seg, int64_t n, const float *n_e, uint64_t seed,
                                float *v, void *workspace, size_t ws_bytes, void *stream)
{
    if (!l || !seg || n < 0 || !v || !workspace || (n > 0 && !n_e)) return LARTPC_ERR_BAD_ARGUMENT;
    if (ws_bytes < lartpc_light_workspace_bytes(l, n)) return LARTPC_ERR_CAPACITY;
    const size_t wf = al256(sizeof(float) * (size_t)l->d.n_det * l->d.n_ticks), sn = al256(sizeof(float) * (size_t)(n ? n : 1));
    unsigned char *b = (unsigned char *)(((uintptr_t)workspace + 255) & ~(uintptr_t)255);
    int32_t *vox = (int32_t *)b;  b += sn;
    int32_t *k0 = (int32_t *)b;  b += sn;
    float *ng = (float *)b;  b += sn;
    float *npe = (float *)b;  b += al256(sizeof(float) * (size_t)l->d.n_det * (size_t)(n ? n : 1));
    float *ipe = (float *)b;  b += wf;
    float *isc = (float *)b;  b += wf;
    float *nobs = (float *)b;
    int rc = lartpc_light_npe(l, seg, n, n_e, vox, k0, ng, npe, stream);
    if (rc == 0) rc = lartpc_light_profile(l, n, vox, k0, npe, ipe, stream);
    if (rc == 0) rc = lartpc_light_scintillation(l, ipe, isc, stream);
    if (rc == 0) rc = lartpc_light_fluctuate(l, seed, isc, nobs, stream);
    if (rc == 0) rc = lartpc_light_electronics(l, seed, nobs, v, stream);
    return rc;
}
