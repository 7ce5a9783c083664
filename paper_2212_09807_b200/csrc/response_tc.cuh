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
// A carries a per-tile power-of-two scale (fp16 range), B a per-LUT one (lartpc_sim_create: max |R| 2^s in (2^9, 2^10], which
// keeps far-field LUT values normal); the fp8 parts carry the extra powers of two below, which cancel in the product; the
// epilogue undoes the rest exactly.
//
// Kernel (persistent, one CTA per SM, 192 threads, whole TMEM):
//   warp 0, one lane   producer: per (item, bin c) one cp.async.bulk per charged 16-tick block of the A image (8 KB each:
//                      fp16 part + fp8 part, un-swizzled K-major, written by charge_lattice_tc_kernel) and one of the Bs
//                      image (14 KB) into a ring of 3 shared-memory stages, completion on an mbarrier per stage
//   warp 1, one lane   MMA issuer: per charged block one fp16 (K = 16) and one fp8 (K = 32) tcgen05.mma (M = 128, N = NBW),
//                      tcgen05.commit frees the stage; after the last bin a commit signals the epilogue
//   warps 2-5          epilogue: tcgen05.ld the fp32 accumulator(s) (thread = tile row), undo the scales, write the
//                      partial waveform rows, zero the accumulator columns again (every MMA accumulates)
// An item is (tile block, row d of the LUT image) -- or TWO neighbouring tile blocks with the same d when each charges at
// most three consecutive 16-tick blocks (tiles are sorted by the blocks they charge, so most do): their accumulators,
// 32 + NBW = 256 columns each counted from the first charged block, share the 512 TMEM columns and every Bs image is
// fetched once for both.  Items are taken from an atomic cursor by the producer (which hands the item to the MMA warp in a
// stage header and from there to the epilogue); consecutive items share their charge blocks, so the CTAs that stream one
// tile block do it at the same time and A is read from HBM once.  (A static round-robin deal lets the CTAs drift apart
// over a long launch: measured, the L2 reuse of A is lost and the kernel becomes HBM-bound.)
#pragma once
#include <cuda_fp16.h>
#include <cuda_fp8.h>
#include <stdint.h>

namespace rtc {

constexpr int TB = 128;            // tiles per tile block (MMA M)
constexpr int JC = 64;             // arrival ticks per tile (K extent per bin): 4 blocks of 16
constexpr int NBLK = JC / 16;
constexpr int STAGES = 3;
constexpr int A_SLOTS = 6;          // charge blocks a stage can hold: 4 of one tile block, or 3 + 3 of a pair
constexpr int THREADS = 192;
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
    int b_scale_log2;              // B = R * 2^b_scale_log2 (DevParams)
    long long n_items;             // ceil(n_tb / 2) * WW * 2: (unit of two tile blocks, row, half)
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

constexpr int stage_bytes(int NBW) { return A_SLOTS * A_BLOCK_BYTES + 2 * NBW * 32; }
constexpr int smem_bytes(int NBW) { return STAGES * stage_bytes(NBW) + 1024 /* alignment slack */ + 256 /* barriers, headers */; }
constexpr int HDR_LAST = 1, HDR_END = 2;
constexpr int PAIR_COL = 256;      // TMEM column of the second accumulator of a pair item

// Two tile blocks share an item -- and with it every LUT generator the item streams -- when each charges at most three
// consecutive 16-tick blocks: an accumulator then needs 32 + NBW <= 256 columns (counted from the block's first charged
// block), and two fit the 512 TMEM columns.
__device__ __forceinline__ bool pairable_mask(int m) { return m != 0 && (31 - __clz(m)) - (__ffs(m) - 1) <= 2; }

// Work items.  Unit u = tile blocks 2u, 2u + 1; cursor value q = (u * rows + d) * 2 + h.  A pairable unit is one item per
// row d (h = 0; h = 1 is skipped); otherwise h picks the tile block.  Consecutive q share their charge blocks.
__global__ void __launch_bounds__(THREADS, 1) response_tc_kernel(const Args a)
{
    extern __shared__ unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int NBW = a.NBW, NC = a.NC;
    const uint32_t b_half = (uint32_t)NBW * 32u;                       // bytes of one precision half of a Bs image
    const uint32_t a_area = (uint32_t)A_SLOTS * A_BLOCK_BYTES;
    const uint32_t stage_sz = a_area + 2u * b_half;                    // multiple of 1024 (NBW multiple of 16)
    const uint32_t base = (s32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bars = base + STAGES * stage_sz;                    // full[S], empty[S], tmem_full, tmem_empty, tmem ptr
    const uint32_t full0 = bars, empty0 = bars + 8 * STAGES, tfull = bars + 16 * STAGES, tempty = tfull + 8;
    const uint32_t titem = tempty + 8, tptr_addr = titem + 8;
    volatile uint32_t *tptr = (volatile uint32_t *)(smem_raw + (tptr_addr - s32(smem_raw)));
    volatile int4 *hdr = (volatile int4 *)(smem_raw + (tptr_addr + 8 - s32(smem_raw)));   // [STAGES] {tbA, d, c | masks, flags}
    volatile int4 *epi_item = hdr + STAGES;                                              // {tbA, d, masks, flags}
    const bool pairs_fit = 32 + NBW <= PAIR_COL;

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
    const int n_acc_cols = 16 * (NBLK - 1) + NBW;                      // columns of a single item's accumulator (272)

    if (warp == 0) {
        // ------------------------------------------------------------------ producer
        if (lane == 0) {
            int s = 0;
            uint32_t ph = 0;
            long long q = atomicAdd(a.work, 1);
            while (q < a.n_items) {
                const long long q_next = atomicAdd(a.work, 1);         // in flight while this item streams
                const int h = (int)(q & 1);
                const long long ud = q >> 1;
                const int u = (int)(ud / a.WW), d = (int)(ud - (long long)u * a.WW);
                const int tb0 = 2 * u, tb1 = tb0 + 1;
                const int m0 = a.tb_mask[tb0] & ((1 << NBLK) - 1), m1 = tb1 < a.n_tb ? a.tb_mask[tb1] & ((1 << NBLK) - 1) : 0;
                const bool pair = pairs_fit && pairable_mask(m0) && pairable_mask(m1);
                int tbA, bmA, bmB = 0;
                if (pair) { tbA = tb0;  bmA = m0;  bmB = m1; }
                else { tbA = h ? tb1 : tb0;  bmA = h ? m1 : m0; }
                if ((pair && h) || bmA == 0) { q = q_next;  continue; }   // the pair went out with h = 0; nothing charged
                const unsigned char *AbA = (const unsigned char *)a.A + (size_t)tbA * NC * (NBLK * A_BLOCK_BYTES);
                const unsigned char *AbB = AbA + (size_t)NC * (NBLK * A_BLOCK_BYTES);   // tile block tbA + 1
                const unsigned char *Bb = (const unsigned char *)a.B + (size_t)d * NC * (2 * b_half);
                const uint32_t a_bytes = (uint32_t)(__popc(bmA) + __popc(bmB)) * A_BLOCK_BYTES;
                for (int c = 0; c < NC; ++c) {
                    mbar_wait(empty0 + 8 * s, ph ^ 1u);
                    const uint32_t st = base + s * stage_sz, fb = full0 + 8 * s;
                    hdr[s].x = tbA;  hdr[s].y = d;  hdr[s].z = c | (bmA << 16) | (bmB << 20);
                    hdr[s].w = (c == NC - 1) ? HDR_LAST : 0;
                    mbar_expect_tx(fb, a_bytes + 2 * b_half);          // release: the header is visible to the waiter
                    uint32_t dst = st;
#pragma unroll
                    for (int b = 0; b < NBLK; ++b)
                        if (bmA >> b & 1) { bulk_g2s(dst, AbA + ((size_t)c * NBLK + b) * A_BLOCK_BYTES, A_BLOCK_BYTES, fb);  dst += A_BLOCK_BYTES; }
#pragma unroll
                    for (int b = 0; b < NBLK; ++b)
                        if (bmB >> b & 1) { bulk_g2s(dst, AbB + ((size_t)c * NBLK + b) * A_BLOCK_BYTES, A_BLOCK_BYTES, fb);  dst += A_BLOCK_BYTES; }
                    bulk_g2s(st + a_area, Bb + (size_t)c * (2 * b_half), 2 * b_half, fb);
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
                const int tbA = hdr[s].x, d = hdr[s].y, cz = hdr[s].z, flags = hdr[s].w;
                const int c = cz & 0xffff, bmA = (cz >> 16) & 15, bmB = (cz >> 20) & 15;
                if (flags & HDR_END) {
                    mbar_wait(tempty, tph);                            // the epilogue has read the previous item slot
                    epi_item->w = HDR_END;
                    mbar_arrive(titem);
                    break;
                }
                if (c == 0) {
                    mbar_wait(tempty, tph);                            // accumulators drained and zeroed
                    epi_item->x = tbA;  epi_item->y = d;  epi_item->z = bmA | (bmB << 4);  epi_item->w = 0;
                    mbar_arrive(titem);                                // release: hands the item to the epilogue
                }
                tc_fence_after();
                const uint32_t st = base + s * stage_sz;
                const uint64_t bd_hi = smem_desc(st + a_area, 128, 256, 0);
                const uint64_t bd_8 = smem_desc(st + a_area + b_half, 128, 256, 0);
                // single item: block b lands at column 16 b; pair: at 16 (b - first charged block) of its own accumulator
                const int lbA = bmB ? __ffs(bmA) - 1 : 0, lbB = bmB ? __ffs(bmB) - 1 : 0;
                uint32_t src = st;
#pragma unroll
                for (int b = 0; b < NBLK; ++b) {
                    if (!(bmA >> b & 1)) continue;                     // no tile of the block has charge in these 16 ticks
                    const uint32_t dcol = tmem + 16 * (b - lbA);
                    tc_mma_f16(dcol, smem_desc(src, 128, 256, 0), bd_hi, idesc, 1u);   // the epilogue leaves the accumulators zero
                    tc_mma_f8(dcol, smem_desc(src + A_PART_BYTES, 128, 256, 0), bd_8, idesc, 1u);
                    src += A_BLOCK_BYTES;
                }
#pragma unroll
                for (int b = 0; b < NBLK; ++b) {
                    if (!(bmB >> b & 1)) continue;
                    const uint32_t dcol = tmem + PAIR_COL + 16 * (b - lbB);
                    tc_mma_f16(dcol, smem_desc(src, 128, 256, 0), bd_hi, idesc, 1u);
                    tc_mma_f8(dcol, smem_desc(src + A_PART_BYTES, 128, 256, 0), bd_8, idesc, 1u);
                    src += A_BLOCK_BYTES;
                }
                tc_commit(empty0 + 8 * s);                             // stage free once these MMAs have read it
                if (flags & HDR_LAST) { tc_commit(tfull); tph ^= 1u; } // accumulators complete
                if (++s == STAGES) { s = 0; ph ^= 1u; }
            }
        }
    } else {
        // ------------------------------------------------------------------ epilogue (warps 2-5)
        const int quad = warp & 3;                                     // TMEM lanes [32 quad, 32 quad + 32)
        const uint32_t tlane = tmem + ((uint32_t)(32 * quad) << 16);
        // every MMA accumulates: the accumulators are zero before the first item and zeroed again after each read-out
        for (int c0 = 0; c0 < 512; c0 += 16) tmem_zero16(tlane + c0);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(tempty);
        uint32_t tph = 0;
        while (true) {
            mbar_wait(titem, tph);                                     // acquire: the MMA warp has published the item
            if (epi_item->w & HDR_END) break;
            const int tbA = epi_item->x, d = epi_item->y, masks = epi_item->z;
            const int bmA = masks & 15, bmB = (masks >> 4) & 15;
            const int n_acc = bmB ? 2 : 1;
            mbar_wait(tfull, tph);
            tc_fence_after();
            for (int x = 0; x < n_acc; ++x) {
                // accumulator x: tile block tbA + x; its column 0 is tick t0 of the tile's window
                const int tile = (tbA + x) * TB + 32 * quad + lane;
                const bool live = tile < a.n_tiles;
                const int t0 = bmB ? 16 * (__ffs(x ? bmB : bmA) - 1) : 0;
                const int n_cols = bmB ? min(PAIR_COL, a.tile_ticks - t0) : a.tile_ticks;     // multiples of 8
                const uint32_t tcol = tlane + (x ? PAIR_COL : 0);
                float scale = 0.f;
                if (live) scale = __int_as_float((127 + a.tile_meta[4 * tile + 2] - a.b_scale_log2) << 23);
                float *dst = a.partial + ((size_t)(live ? tile : 0) * a.WW + d) * a.tile_ticks + t0;
                if (bmB && live) {
                    // S5 reads whole 14-tick blocks around the charged range: the few ticks of the row the accumulator
                    // does not cover (before the first charged block, after column 255) are zero
                    float *row = dst - t0;
                    for (int i = 0; i < t0; i += 4) __stcs((float4 *)(row + i), make_float4(0.f, 0.f, 0.f, 0.f));
                    for (int i = t0 + n_cols; i < a.tile_ticks; i += 4) __stcs((float4 *)(row + i), make_float4(0.f, 0.f, 0.f, 0.f));
                }
                const int n_full = n_cols / 32;
                for (int ch = 0; ch < n_full; ++ch) {
                    uint32_t v[32];
                    tmem_ld32(tcol + 32 * ch, v);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (live) {
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            __stcs((float4 *)(dst + 32 * ch) + i, make_float4(__uint_as_float(v[4 * i]) * scale, __uint_as_float(v[4 * i + 1]) * scale,
                                                                         __uint_as_float(v[4 * i + 2]) * scale, __uint_as_float(v[4 * i + 3]) * scale));
                    }
                }
                for (int c0 = 32 * n_full; c0 < n_cols; c0 += 8) {
                    uint32_t v[8];
                    tmem_ld8(tcol + c0, v);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (live) {
#pragma unroll
                        for (int i = 0; i < 2; ++i)
                            __stcs((float4 *)(dst + c0) + i, make_float4(__uint_as_float(v[4 * i]) * scale, __uint_as_float(v[4 * i + 1]) * scale,
                                                                    __uint_as_float(v[4 * i + 2]) * scale, __uint_as_float(v[4 * i + 3]) * scale));
                    }
                }
            }
            const int n_zero = bmB ? 512 : n_acc_cols;
            for (int c0 = 0; c0 < n_zero; c0 += 16) tmem_zero16(tlane + c0);
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
