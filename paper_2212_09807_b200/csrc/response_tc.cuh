// S4 response on the 5th-generation tensor cores (tcgen05 + TMEM), eq. (3.7) P:L660-665 as a dense contraction.
//
// For one tile t (charged pixel, window of Jc = 64 arrival ticks) and one target pixel d of the W x W window,
//     I_d[n] = sum_c sum_j C_t[c][j] R[c][d][n - j]                    c: LUT bin, j: arrival tick, n: readout tick
// is a row of the matrix product  D = A B  with A[t][(c, j)] = C_t[c][j] (128 tiles per CTA = the M dimension) and
// the Toeplitz matrix B[(c, j)][n] = R[c][d][n - j].  Writing j = 16 b + jj, the block of B for arrival ticks
// [16 b, 16 b + 16) is the SAME matrix Bs[c][jj][n'] = R[c][d][n' - jj] shifted by 16 b output columns, so one
// 16 x NBW operand (NBW = roundup16(K + 15) = 224 for K = 200) serves all four b: the MMA for block b accumulates
// into TMEM columns [16 b, 16 b + NBW).  Bs for all (d, c) is 36 MB and stays in L2; nothing Toeplitz-sized is built.
//
// Precision: tensor-core inputs are fp16, so both operands are split x = hi + lo (hi = fp16(x), lo = x - hi) and
// hi*hi + hi*lo + lo*hi is accumulated in fp32 (the dropped lo*lo term is 2^-22 relative).  The two cross terms are
// 2^-11 of the main one, so three significant bits are all they need: they run as ONE fp8 (e4m3) MMA of K = 32,
//     [lo8(A) | hi8(A)] x [hi8(B) ; lo8(B)],
// which costs the tensor pipe as much as one fp16 MMA of K = 16: two MMA slots per (bin, 16-tick block) instead of three
// (error of the cross terms: 2^-4 x 2^-12 relative per product, random in sign; parity margins in the tests unchanged).
// A carries a per-tile power-of-two scale (fp16 range), B a fixed 2^10 (keeps far-field LUT values normal); the fp8
// parts carry the extra powers of two below, which cancel in the product; the epilogue undoes the rest exactly.
//
// Kernel (persistent, one CTA per SM, 192 threads, whole TMEM):
//   warp 0, one lane   producer: per (item = (tile block, d), bin c) one cp.async.bulk of the A image (hi + lo, 32 KB,
//                      written by charge_lattice_kernel already in the 128-byte-swizzled K-major UMMA layout) and one of
//                      the Bs image (hi + lo, 14 KB, canonical un-swizzled K-major layout built at create) into a ring
//                      of 4 shared-memory stages, completion on an mbarrier per stage
//   warp 1, one lane   MMA issuer: 8 tcgen05.mma (M = 128, N = NBW; 4 blocks b x (fp16 K = 16 + fp8 K = 32)) per
//                      stage, tcgen05.commit frees the stage; after the last bin a commit signals the epilogue
//   warps 2-5          epilogue: tcgen05.ld the 128 x 264 fp32 accumulator (thread = tile row), undo the scales, write
//                      the partial waveform rows, re-zero the TMEM columns that only later blocks b touch
// Items are taken from an atomic cursor by the producer (which hands the item to the MMA warp in a stage header and
// from there to the epilogue), consecutive items share the tile block, so the 25 CTAs that stream one A block do it at
// the same time and A is read from HBM once.  (A static round-robin deal lets the CTAs drift apart over a long
// launch: measured, the L2 reuse of A is lost and the kernel becomes HBM-bound.)
#pragma once
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <stdint.h>

namespace rtc {

constexpr int TB = 128;            // tiles per tile block (MMA M)
constexpr int JC = 64;             // arrival ticks per tile (K extent per bin): 4 blocks of 16
constexpr int NBLK = JC / 16;
constexpr int STAGES = 4;
constexpr int THREADS = 192;
constexpr int B_SCALE_LOG2 = 10;
// fp8 parts: lo8(A) = e4m3(lo(A) 2^SA) meets hi8(B) = e4m3(B 2^-SA); hi8(A) = e4m3(A 2^-SB) meets lo8(B) = e4m3(lo(B) 2^SB)
// (|A| < 2^15, |lo(A)| <= 8, |B| <= 2^10, |lo(B)| <= 0.5: every part stays below e4m3's 448)
constexpr int SA_LOG2 = 5, SB_LOG2 = 7;
constexpr int A_HALF_BYTES = TB * JC * 2;          // half of a stage's A area (the area holds NBLK blocks of 8 KB)

struct Args {
    const __half *A;               // [n_tb][NC][2][TB][128 bytes]: fp16 image (a_image_offset) + fp8 image (a8_image_offset)
    const __half *B;               // [WW][NC][2][NBW * 32 bytes]: fp16 image (b_image_offset) + fp8 image (b8_image_offset)
    float *partial;                // [n_tiles][WW][tile_ticks]
    const int32_t *tile_meta;      // [n_tiles][4]: first / last output block, scale exponent e (A = C * 2^-e), 0
    const int32_t *tb_mask;        // [n_tb] 16-tick blocks that hold charge in any tile of the block (bit b)
    int n_tiles, n_tb, NC, WW, NBW, tile_ticks;
    long long n_items;             // n_tb * WW
    int *work;                     // item cursor, zero at launch: items are taken in order as CTAs become free, so the
                                   // CTAs that stream one tile block stay together however long the launch runs
};

// A image: [tile block][bin c][16-tick block b][fp16 part | fp8 part][128 rows x 32 bytes], each part a canonical
// un-swizzled K-major operand of one MMA (row r = tile in block; 16-byte K chunks 128 B apart, 8-row groups 256 B apart),
// so that a stage copies only the 16-tick blocks that hold charge.  Byte offset of K chunk kc (0 / 1) of row r in a part:
__host__ __device__ __forceinline__ int a_part_offset(int r, int kc) { return (r >> 3) * 256 + kc * 128 + (r & 7) * 16; }
constexpr int A_PART_BYTES = 128 * 32;                 // one part of one block: 4 KB
constexpr int A_BLOCK_BYTES = 2 * A_PART_BYTES;        // fp16 part + fp8 part
// canonical un-swizzled K-major image of Bs: row n' (output column), element jj: 8 x 16-byte core matrices,
// K chunks 128 B apart (LBO), 8-row groups 256 B apart (SBO)
__host__ __device__ __forceinline__ int b_image_offset(int n, int jj)         // in halfs
{
    return (n >> 3) * 128 + (jj >> 3) * 64 + (n & 7) * 8 + (jj & 7);
}

// fp8 image of Bs: row n', K byte kb in [0, 32): kb < 16 -> hi8 of jj = kb, else lo8 of jj = kb - 16; same canonical
// K-major byte layout as the fp16 image (16-byte core rows, K chunks 128 B apart, 8-row groups 256 B apart)
__host__ __device__ __forceinline__ int b8_image_offset(int n, int kb)
{
    return (n >> 3) * 256 + (kb >> 4) * 128 + (n & 7) * 16 + (kb & 15);
}

// Writes 16 consecutive arrival ticks (one block b) of row r of one bin's A operand: x = C 2^-e, |x| < 2^15.
// blk: start of that (bin, block) in the image (A_BLOCK_BYTES).  fp16 part: ticks 0-7 | 8-15; fp8 part: lo8 | hi8.
__device__ __forceinline__ void store_a_block16(unsigned char *blk, int r, const float (&x)[16])
{
    __half2 h[8];
    unsigned short l8[8], h8[8];
    const float sa = (float)(1 << SA_LOG2), sb = 1.0f / (float)(1 << SB_LOG2);
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        h[i] = __floats2half2_rn(x[2 * i], x[2 * i + 1]);
        const float2 f = __half22float2(h[i]);
        l8[i] = __nv_cvt_float2_to_fp8x2(make_float2((x[2 * i] - f.x) * sa, (x[2 * i + 1] - f.y) * sa), __NV_SATFINITE, __NV_E4M3);
        h8[i] = __nv_cvt_float2_to_fp8x2(make_float2(x[2 * i] * sb, x[2 * i + 1] * sb), __NV_SATFINITE, __NV_E4M3);
    }
    const int o0 = a_part_offset(r, 0), o1 = a_part_offset(r, 1);
    *(uint4 *)(blk + o0) = *(const uint4 *)&h[0];
    *(uint4 *)(blk + o1) = *(const uint4 *)&h[4];
    *(uint4 *)(blk + A_PART_BYTES + o0) = *(const uint4 *)l8;
    *(uint4 *)(blk + A_PART_BYTES + o1) = *(const uint4 *)h8;
}

__device__ __forceinline__ uint32_t s32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_mma_f16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}
__device__ __forceinline__ void tc_mma_f8(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "setp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n"
        "}\n" ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc) : "memory");
}
// shared-memory matrix descriptor (version 1): start address, leading / stride byte offsets in 16-byte units, layout
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes, uint32_t layout)
{
    return (uint64_t)((addr >> 4) & 0x3FFFu) | ((uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16) |
           ((uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32) | (1ull << 46) | ((uint64_t)layout << 61);
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
          "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
          "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&v)[8])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_zero16(uint32_t taddr)
{
    const uint32_t z = 0u;
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], "
        "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};\n" ::"r"(taddr), "r"(z) : "memory");
}

constexpr int stage_bytes(int NBW) { return 2 * A_HALF_BYTES + 2 * NBW * 32; }
constexpr int smem_bytes(int NBW) { return STAGES * stage_bytes(NBW) + 1024 /* alignment slack */ + 256 /* barriers, headers */; }
constexpr int HDR_LAST = 1, HDR_END = 2;

__global__ void __launch_bounds__(THREADS, 1) response_tc_kernel(const Args a)
{
    extern __shared__ unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NBW = a.NBW, NC = a.NC;
    const uint32_t b_half = (uint32_t)NBW * 32u;                       // bytes of one precision half of a Bs image
    const uint32_t stage_sz = 2u * A_HALF_BYTES + 2u * b_half;         // multiple of 1024 (NBW multiple of 16)
    // SWIZZLE_128B operands need 1024-byte aligned tiles
    const uint32_t base = (s32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bars = base + STAGES * stage_sz;                    // full[S], empty[S], tmem_full, tmem_empty, tmem ptr
    const uint32_t full0 = bars, empty0 = bars + 8 * STAGES, tfull = bars + 16 * STAGES, tempty = tfull + 8;
    const uint32_t titem = tempty + 8, tptr_addr = titem + 8;
    volatile uint32_t *tptr = (volatile uint32_t *)(smem_raw + (tptr_addr - s32(smem_raw)));
    volatile int4 *hdr = (volatile int4 *)(smem_raw + (tptr_addr + 8 - s32(smem_raw)));   // [STAGES] {tb, d, c, flags}
    volatile int4 *epi_item = hdr + STAGES;                                              // {tb, d, 0, flags}

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
        mbar_init(tfull, 1);
        mbar_init(tempty, 4);                                          // one arrival per epilogue warp
        mbar_init(titem, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {                                                   // the MMA warp owns the TMEM allocation
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tptr_addr), "r"(512u) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tptr;
    const int n_acc_cols = 16 * (NBLK - 1) + NBW;                      // accumulator columns in use (272)

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            long long q = atomicAdd(a.work, 1);
            while (q < a.n_items) {
                const long long q_next = atomicAdd(a.work, 1);         // in flight while this item streams
                const int tb = (int)(q / a.WW), d = (int)(q - (long long)tb * a.WW);
                const unsigned char *Ab = (const unsigned char *)a.A + (size_t)tb * NC * (2 * A_HALF_BYTES);
                const unsigned char *Bb = (const unsigned char *)a.B + (size_t)d * NC * (2 * b_half);
                const int bm = a.tb_mask[tb] & ((1 << NBLK) - 1);
                const uint32_t a_bytes = (uint32_t)__popc(bm) * A_BLOCK_BYTES;
                for (int c = 0; c < NC && bm; ++c) {
                    mbar_wait(empty0 + 8 * s, ph ^ 1u);
                    const uint32_t st = base + s * stage_sz, fb = full0 + 8 * s;
                    hdr[s].x = tb;  hdr[s].y = d;  hdr[s].z = c | (bm << 16);  hdr[s].w = (c == NC - 1) ? HDR_LAST : 0;
                    mbar_expect_tx(fb, a_bytes + 2 * b_half);          // release: the header is visible to the waiter
                    const unsigned char *Ac = Ab + (size_t)c * (NBLK * A_BLOCK_BYTES);
#pragma unroll
                    for (int b = 0; b < NBLK; ++b)
                        if (bm >> b & 1) bulk_g2s(st + b * A_BLOCK_BYTES, Ac + b * A_BLOCK_BYTES, A_BLOCK_BYTES, fb);
                    bulk_g2s(st + 2 * A_HALF_BYTES, Bb + (size_t)c * (2 * b_half), 2 * b_half, fb);
                    if (++s == STAGES) { s = 0; ph ^= 1u; }
                }
                q = q_next;
            }
            mbar_wait(empty0 + 8 * s, ph ^ 1u);                        // terminator: a header-only stage
            hdr[s].w = HDR_END;
            mbar_arrive(full0 + 8 * s);
        }
    } else if (warp == 1) {
        // ------------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            // instruction descriptor: D fp32, A and B fp16 (kind::f16) or e4m3 (kind::f8f6f4) -- format code 0 in both
            // kinds --, both K-major, N = NBW, M = 128
            const uint32_t idesc = (1u << 4) | ((uint32_t)(NBW >> 3) << 17) | ((uint32_t)(TB >> 4) << 24);
            int s = 0;
            uint32_t ph = 0, tph = 0;
            while (true) {
                mbar_wait(full0 + 8 * s, ph);
                const int tb = hdr[s].x, d = hdr[s].y, cz = hdr[s].z, flags = hdr[s].w;
                const int c = cz & 0xffff, bm = cz >> 16;
                if (flags & HDR_END) {
                    mbar_wait(tempty, tph);                            // the epilogue has read the previous item slot
                    epi_item->w = HDR_END;
                    mbar_arrive(titem);
                    break;
                }
                if (c == 0) {
                    mbar_wait(tempty, tph);                            // accumulator drained and zeroed
                    epi_item->x = tb;  epi_item->y = d;  epi_item->w = 0;
                    mbar_arrive(titem);                                // release: hands the item to the epilogue
                }
                tc_fence_after();
                const uint32_t st = base + s * stage_sz;
                const uint64_t bd_hi = smem_desc(st + 2 * A_HALF_BYTES, 128, 256, 0);
                const uint64_t bd_8 = smem_desc(st + 2 * A_HALF_BYTES + b_half, 128, 256, 0);
#pragma unroll
                for (int b = 0; b < NBLK; ++b) {
                    if (!(bm >> b & 1)) continue;                      // no tile of the block has charge in these 16 ticks
                    const uint64_t ad_hi = smem_desc(st + b * A_BLOCK_BYTES, 128, 256, 0);
                    const uint64_t ad_8 = smem_desc(st + b * A_BLOCK_BYTES + A_PART_BYTES, 128, 256, 0);
                    const uint32_t dcol = tmem + 16 * b;
                    tc_mma_f16(dcol, ad_hi, bd_hi, idesc, 1u);         // the epilogue leaves the whole accumulator zero
                    tc_mma_f8(dcol, ad_8, bd_8, idesc, 1u);
                }
                tc_commit(empty0 + 8 * s);                             // stage free once these MMAs have read it
                if (flags & HDR_LAST) { tc_commit(tfull); tph ^= 1u; } // accumulator complete
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue (warps 2-5)
        const int quad = warp & 3;                                     // TMEM lanes [32 quad, 32 quad + 32)
        const uint32_t tlane = tmem + ((uint32_t)(32 * quad) << 16);
        // every MMA accumulates: the accumulator is zero before the first item and zeroed again after each read-out
        for (int c0 = 0; c0 < n_acc_cols; c0 += 16) tmem_zero16(tlane + c0);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty);
        uint32_t tph = 0;
        const int n_full = a.tile_ticks / 32, n_rem = a.tile_ticks - 32 * n_full;   // tile_ticks = 264: 8 x 32 + 8
        while (true) {
            mbar_wait(titem, tph);                                     // acquire: the MMA warp has published the item
            if (epi_item->w & HDR_END) break;
            const int tb = epi_item->x, d = epi_item->y;
            const int tile = tb * TB + 32 * quad + lane;
            const bool live = tile < a.n_tiles;
            float scale = 0.f;
            if (live) scale = __int_as_float((127 + a.tile_meta[4 * tile + 2] - B_SCALE_LOG2) << 23);
            float *dst = a.partial + ((size_t)(live ? tile : 0) * a.WW + d) * a.tile_ticks;
            mbar_wait(tfull, tph);
            tc_fence_after();
            for (int ch = 0; ch < n_full; ++ch) {
                uint32_t v[32];
                tmem_ld32(tlane + 32 * ch, v);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (live) {
#pragma unroll
                    for (int i = 0; i < 8; ++i)
                        __stcs((float4 *)(dst + 32 * ch) + i, make_float4(__uint_as_float(v[4 * i]) * scale, __uint_as_float(v[4 * i + 1]) * scale,
                                                                     __uint_as_float(v[4 * i + 2]) * scale, __uint_as_float(v[4 * i + 3]) * scale));
                }
            }
            if (n_rem) {
                uint32_t v[8];
                tmem_ld8(tlane + 32 * n_full, v);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (live) {
#pragma unroll
                    for (int i = 0; i < 2; ++i)
                        __stcs((float4 *)(dst + 32 * n_full) + i, make_float4(__uint_as_float(v[4 * i]) * scale, __uint_as_float(v[4 * i + 1]) * scale,
                                                                         __uint_as_float(v[4 * i + 2]) * scale, __uint_as_float(v[4 * i + 3]) * scale));
                }
            }
            for (int c0 = 0; c0 < n_acc_cols; c0 += 16) tmem_zero16(tlane + c0);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty);
            tph ^= 1u;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}

}  // namespace rtc
