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
#ifndef LARTPC_EPI_GROUPS
#define LARTPC_EPI_GROUPS 1
#endif
// An item's read-out (TMEM -> registers -> HBM) sits between two items' MMAs: the accumulators are single.  EPI_G warps per
// TMEM lane quarter share its column chunks; measured at configs[3], 1 -> 2 -> 4 warps shorten it 7 700 -> 6 600 -> 6 500
// cycles (TMEM reads at 64 B / cycle: 3 800 cycles for the two accumulators) and leave the kernel's time where it was
// (profiles/r2_response_bound.md), so one warp per quarter it stays.
constexpr int EPI_G = LARTPC_EPI_GROUPS;
// warps: producer, MMA issuer (even blocks) / relay, 4 x epilogue, MMA issuer (odd blocks), 4 x epilogue per further group
constexpr int THREADS = 224 + 128 * (EPI_G - 1);
// fp8 parts: lo8(A) = e4m3(lo(A) 2^SA) meets hi8(B) = e4m3(B 2^-SA); hi8(A) = e4m3(A 2^-SB) meets lo8(B) = e4m3(lo(B) 2^SB)
// (|A| < 2^15, |lo(A)| <= 8, |B| <= 2^10, |lo(B)| <= 0.5: every part stays below e4m3's 448)
constexpr int SA_LOG2 = 5, SB_LOG2 = 7;

struct Args {
    const __half *A;               // [n_tb][NC][2][TB][128 bytes]: fp16 image (a_image_offset) + fp8 image (a8_image_offset)
    const __half *B;               // [WW][NC][CTA of the pair][fp16 image (b_image_offset) | fp8 image (b8_image_offset)] of that CTA's rows
    float *partial;                // [n_tiles][WW][tile_ticks]
    const int32_t *tile_meta;      // [n_tiles][4]: first / last output block, scale exponent e (A = C * 2^-e), non-zero cells
                                   // per 16-tick block / 8 (one byte per block)
    const int32_t *tb_mask;        // [n_units] 16-tick blocks that hold charge in any tile of the unit (bit b)
    const int32_t *cmask;          // [n_units][CMW] per bin (4 bits, 8 bins per word) the blocks some tile of the unit charges
    int n_tiles, n_units, NC, WW, NBW, tile_ticks, n_stages;
    int b_scale_log2;              // B = R * 2^b_scale_log2 (DevParams)
    int K;                         // LUT ticks of a row (whole LUT, or one piece of it)
    float kappa;                   // expected relative truncation loss per accumulated product (see "Accuracy"), 0 = off
    long long n_items;             // n_units * WW: (unit, row of the LUT image)
    unsigned long long *stats;     // device counters (lartpc_get_counters): [1] MMAs issued, [2] bytes copied, [5] items
    int *work;                     // item cursor, zero at launch: items are taken in order as CTAs become free, so the
                                   // CTAs that stream one tile block stay together however long the launch runs
};

// A image: [tile block][bin c][16-tick block b][fp16 part | fp8 part][128 rows x 32 bytes], each part a K-major operand of
// one MMA in the 32-byte-swizzle canonical layout (row r = tile in block; a row's 32 bytes are contiguous, 8-row groups
// 256 B apart), so that a stage copies only the 16-tick blocks that hold charge AND a tile's row is a whole 32-byte DRAM
// sector: with the un-swizzled layout (16-byte pieces, two rows per sector, written by different CTAs at different times)
// the charge lattice wrote every sector twice and read it back once in between (profiles/r2_traffic_c3.md).
// Byte offset of K chunk kc (0 / 1) of row r in a part:
// (32-byte swizzle atom: 8 rows x 32 bytes, the two 16-byte K chunks of rows 4-7 swapped -- address bit 7 XORed into bit 4)
__host__ __device__ __forceinline__ int a_part_offset(int r, int kc) { return (r >> 3) * 256 + (r & 7) * 32 + ((kc ^ ((r >> 2) & 1)) * 16); }
constexpr uint32_t A_LAYOUT = 6;                        // UMMA descriptor layout type SWIZZLE_32B
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

__device__ __forceinline__ void st_global_256(void *p, const uint4 &a, const uint4 &b)     // 32-byte aligned
{
    // evict-first: the operand image (57 GB per configs[3] spill) and the partial rows (82 GB) are read back long after they
    // have left the 126 MB L2; not letting them push the LUT images and the operand blocks in use out of it is worth 1 - 2 ms
    asm volatile("st.global.cs.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};"
                 ::"l"(p), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w) : "memory");
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
    // a row of a part is one 32-byte sector: one 256-bit store each (the two K chunks swapped in rows 4-7 of an atom)
    const bool sw = (r >> 2) & 1;
    const uint4 c0 = *(const uint4 *)&h[0], c1 = *(const uint4 *)&h[4], d0 = *(const uint4 *)l8, d1 = *(const uint4 *)h8;
    st_global_256(blk + a_part_offset(r, sw ? 1 : 0), sw ? c1 : c0, sw ? c0 : c1);
    st_global_256(blk + A_PART_BYTES + a_part_offset(r, sw ? 1 : 0), sw ? d1 : d0, sw ? d0 : d1);
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
__device__ __forceinline__ void tmem_zero64(uint32_t taddr)
{
    const uint32_t z = 0u;
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x64.b32 [%0], "
        "{%1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1, %1};\n" ::"r"(taddr), "r"(z) : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}

// ---- cluster (CTA pair) helpers -----------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
// shared::cluster address of `addr` (a shared::cta address of this CTA) in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t mapa(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)       // acquire at cluster scope
{
    uint32_t ok = 0;
    while (!ok) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    }
}
// remote arrive that orders nothing but the barrier itself (what it reports was written by the async proxy and is
// read by the async proxy)
__device__ __forceinline__ void mbar_arrive_remote_relaxed(uint32_t cluster_bar)
{
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_bar)
{
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_remote(uint32_t cluster_bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.release.cluster.shared::cluster.b64 _, [%0], %1;" ::"r"(cluster_bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void st_cluster_v4(uint32_t cluster_addr, int x, int y, int z, int w)
{
    asm volatile("st.shared::cluster.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(cluster_addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
template <bool CTA2> __device__ __forceinline__ void tc_mma(bool f8, uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc)
{
    // every MMA accumulates (the epilogue leaves the accumulators zero)
    if (CTA2) {
        if (f8) asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, 1, 0;\ntcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n}\n"
                             ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc) : "memory");
        else asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, 1, 0;\ntcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n}\n"
                          ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc) : "memory");
    } else {
        if (f8) tc_mma_f8(d_tmem, a_desc, b_desc, idesc, 1u);
        else tc_mma_f16(d_tmem, a_desc, b_desc, idesc, 1u);
    }
}
// commit of everything this thread has issued so far: arrive on `bar` of this CTA, or (cta_mask) of both CTAs of the pair
template <bool CTA2> __device__ __forceinline__ void tc_commit_x(uint32_t bar, bool both)
{
    if (!CTA2) { tc_commit(bar); return; }
    if (both) {
        const unsigned short mask = 3;
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                     ::"r"(bar), "h"(mask) : "memory");
    } else {
        asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
    }
}

#ifdef LARTPC_DEBUG_CLOCKS
__device__ unsigned long long g_rtc_dbg[16];   // measurement build: cycles the MMA issuer / producer spend per phase
#define RTC_T(x) const long long x = clock64()
#define RTC_DECL unsigned long long rtc_acc[16] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0}
#define RTC_ADD(i, v) rtc_acc[i] += (unsigned long long)(v)                 // per thread; one flush when the role ends
#define RTC_FLUSH do { for (int i_ = 0; i_ < 16; ++i_) if (rtc_acc[i_]) atomicAdd(&g_rtc_dbg[i_], rtc_acc[i_]); } while (0)
#else
#define RTC_T(x)
#define RTC_DECL
#define RTC_ADD(i, v)
#define RTC_FLUSH
#endif
constexpr int MAX_STAGES = 8;
constexpr int N_MAIL = MAX_STAGES + 2;  // item mailbox slots of the peer: the leader's producer is never more than a ring ahead
constexpr int HDR_FIRST = 1, HDR_LAST = 2, HDR_END = 4;
constexpr int ACC_COL = 256;       // TMEM column of the second accumulator (odd 16-tick blocks)
constexpr int CMW = 16;            // words of a unit's per-bin block mask (common.cuh TC_CMASK_WORDS)

// bytes of Bs one CTA holds per (target, bin): both precision parts of all rows, or of half the rows with the CTA pair
__host__ __device__ inline uint32_t b_cta_bytes(int NBW, bool cta2) { return (uint32_t)(cta2 ? NBW * 32 : NBW * 64); }
// a stage = the A blocks of one bin (up to NBLK, 8 KB each: fp16 + fp8 part) + this CTA's rows of the bin's generator
__host__ __device__ inline uint32_t stage_bytes(int NBW, bool cta2)
{
    return (uint32_t)((NBLK * A_BLOCK_BYTES + b_cta_bytes(NBW, cta2) + 1023) & ~1023);
}
inline int n_stages(int NBW, bool cta2, size_t smem_limit)
{
    const int n = (int)((smem_limit - 3072) / stage_bytes(NBW, cta2));
    return n > MAX_STAGES ? MAX_STAGES : n;
}
inline size_t smem_bytes(int NBW, bool cta2, int stages) { return (size_t)stages * stage_bytes(NBW, cta2) + 1024 /* alignment */ + 2048 /* barriers, headers */; }

// Work item = (unit u, row d of the LUT image).  Cursor value q = u * rows + d: consecutive items share their charge
// blocks, and the CTAs that stream one unit do it at about the same time, so A comes from HBM once.
//
// Roles (192 threads per CTA; with CTA2 the kernel runs as clusters of two CTAs on one TPC, rank 0 = leader):
//   warp 0, one lane   producer, in every CTA, filling its own shared memory with its own TMA engine (copies into the
//                      partner's memory would cross the SM-to-SM network at a fraction of the rate).  One stage per
//                      (item, bin c): the A blocks (fp16 + fp8 part) of the charged 16-tick blocks of this CTA's tile
//                      block -- ONE bulk copy per run of consecutive charged blocks, they are neighbours in the image --
//                      and this CTA's rows of the generator, one more copy (the LUT image is laid out per CTA of the pair).
//                      The issue rate of cp.async.bulk by one thread is what bounds the kernel otherwise (measured:
//                      ~250 cycles per copy).  The leader takes the items from the cursor and posts each item's header
//                      in the peer's mailbox, one message per item; after that the two producers run on their own,
//                      paced by their own empty barriers (the MMA issuer's commits arrive in both CTAs).
//   warp 1, one lane   leader: MMA issuer.  Per stage: waits full (and pfull: the peer's share has landed), issues the
//                      fp16 and the fp8 tcgen05.mma of every charged block (M = 128, or 256 over the pair with
//                      cta_group::2: each CTA multiplies its own 128 tiles by the whole generator, of which it holds half
//                      the rows), commits empty; after an item's last stage tfull, in both CTAs.
//                      peer: relay.  Waits its own full and arrives on the leader's pfull.
//   warps 2-5          epilogue, every CTA: adds the two accumulators, undoes the scales, writes the partial rows of
//                      its own tile block, zeroes the accumulators, arrives on the leader's tempty.
// Accuracy.  tcgen05.mma adds into the fp32 accumulator with truncation (toward zero: measured), so a long accumulation
// chain loses a fraction of an ulp per product, systematically.  Even and odd 16-tick blocks therefore accumulate into
// separate accumulators (columns [0, 256) and [256, 512): block b at column 32 (b / 2) of accumulator b % 2), which the
// epilogue adds in round-to-nearest: half as many products per accumulator.
template <bool CTA2>
__global__ void __launch_bounds__(THREADS, 1) response_tc_kernel(const Args a)
{
    extern __shared__ unsigned char smem_raw[];
    __shared__ uint32_t s_cm[CMW];                                     // producer: the current unit's per-bin block masks
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t rank = CTA2 ? cluster_ctarank() : 0u;
    const bool leader = rank == 0u;
    const int NBW = a.NBW, NC = a.NC, S = a.n_stages;
    const uint32_t b_cta = b_cta_bytes(NBW, CTA2);                     // this CTA's rows of a generator: fp16 part, fp8 part
    const uint32_t a_area = (uint32_t)NBLK * A_BLOCK_BYTES;
    const uint32_t stage_sz = stage_bytes(NBW, CTA2);
    const uint32_t base = (s32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bars = base + (uint32_t)S * stage_sz;
    const uint32_t full0 = bars, empty0 = full0 + 8 * MAX_STAGES, pfull0 = empty0 + 8 * MAX_STAGES;
    const uint32_t gox0 = pfull0 + 8 * MAX_STAGES;
    const uint32_t tfull = gox0 + 8 * N_MAIL, tempty = tfull + 8, titem = tempty + 8, tptr_addr = titem + 8;
    const uint32_t hdr0 = (tptr_addr + 8 + 15u) & ~15u, epi0 = hdr0 + 16 * MAX_STAGES, mail0 = epi0 + 16;
    unsigned char *gen = smem_raw - s32(smem_raw);                     // shared::cta address -> generic pointer
    volatile uint32_t *tptr = (volatile uint32_t *)(gen + tptr_addr);
    volatile int4 *hdr = (volatile int4 *)(gen + hdr0);                // [S] {unit, d, c | mask << 16, flags}
    volatile int4 *epi_item = (volatile int4 *)(gen + epi0);           // {unit, d, mask, flags}

    if (tid == 0) {
        // empty[s] and tfull take one commit from each of the two MMA issuers
        for (int s = 0; s < S; ++s) { mbar_init(full0 + 8 * s, 1);  mbar_init(empty0 + 8 * s, 2);  mbar_init(pfull0 + 8 * s, 1); }
        for (int m = 0; m < N_MAIL; ++m) mbar_init(gox0 + 8 * m, 1);
        mbar_init(tfull, 2);
        mbar_init(tempty, (CTA2 ? 8 : 4) * EPI_G);                     // one arrival per epilogue warp of the pair
        mbar_init(titem, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {                                                   // warp 1 of every CTA owns its TMEM allocation
        if (CTA2) {
            asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tptr_addr), "r"(512u) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
        } else {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tptr_addr), "r"(512u) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
    }
    tc_fence_before();
    __syncthreads();
    if (CTA2) cluster_sync_all();                                      // barriers and TMEM of both CTAs exist
    tc_fence_after();
    const uint32_t tmem = *tptr;

    if (warp == 0) {
        if (lane == 0) {
            // ------------------------------------------------------------------ producer (leader: schedules; peer: follows)
            RTC_DECL;
            const uint32_t peer_gox0 = CTA2 ? mapa(gox0, 1u) : 0u, peer_mail0 = CTA2 ? mapa(mail0, 1u) : 0u;
            volatile int4 *mail = (volatile int4 *)(gen + mail0);
            const size_t tb_stride = (size_t)NC * (NBLK * A_BLOCK_BYTES);
            const size_t b_stride = (size_t)(CTA2 ? 2 : 1) * b_cta;    // one (target, bin) of the LUT image: [CTA of the pair][fp16 | fp8]
            int s = 0, m = 0;
            uint32_t ph = 0, mph = 0;
            long long q = leader ? atomicAdd(a.work, 1) : 0;
            while (true) {
                int u, d, mask;
                long long q_next = 0;
                if (leader) {
                    const bool end = q >= a.n_items;
                    u = d = mask = 0;
                    if (!end) {
                        q_next = atomicAdd(a.work, 1);                 // in flight while this item streams
                        u = (int)(q / a.WW);  d = (int)(q - (long long)u * a.WW);
                        mask = a.tb_mask[u] & ((1 << NBLK) - 1);
                        if (mask == 0) { q = q_next;  continue; }      // nothing charged
                    }
                    if (CTA2) { st_cluster_v4(peer_mail0 + 16 * m, u, d, mask, end ? HDR_END : 0);  mbar_arrive_remote(peer_gox0 + 8 * m); }
                    if (end) break;
                } else {
                    mbar_wait_cluster(gox0 + 8 * m, mph);
                    if (mail[m].w & HDR_END) break;
                    u = mail[m].x;  d = mail[m].y;  mask = mail[m].z;
                }
                if (++m == N_MAIL) { m = 0; mph ^= 1u; }
                const unsigned char *Ab = (const unsigned char *)a.A + ((size_t)u * (CTA2 ? 2 : 1) + rank) * tb_stride;
                const unsigned char *Bd = (const unsigned char *)a.B + (size_t)d * NC * b_stride + (size_t)rank * b_cta;
                // per bin the blocks some tile of the unit charges: a (bin, block) pair nobody charges is neither copied nor
                // multiplied, a bin nobody charges takes no stage at all
                int c_first = -1, c_last = -1;
                {
                    const uint4 *src = (const uint4 *)(a.cmask + (size_t)u * CMW);
#pragma unroll
                    for (int w4 = 0; w4 < CMW / 4; ++w4) {
                        const uint4 x = __ldg(src + w4);
                        const uint32_t xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                        for (int k = 0; k < 4; ++k) {
                            const int w = 4 * w4 + k;
                            // keep only the blocks of the unit's mask, bin by bin (a nibble each), and the bins that exist
                            uint32_t v = xs[k] & ((uint32_t)mask * 0x11111111u);
                            if (8 * w >= NC) v = 0u;
                            else if (8 * w + 8 > NC) v &= (1u << (4 * (NC - 8 * w))) - 1u;
                            if (v) { if (c_first < 0) c_first = 8 * w + ((__ffs(v) - 1) >> 2);  c_last = 8 * w + ((31 - __clz(v)) >> 2); }
                            s_cm[w] = v;                               // (this thread's own scratch)
                        }
                    }
                }
                if (c_first < 0) { q = q_next;  continue; }                // (CTA2: the peer computes the same and skips too)
                unsigned long long n_mma = 0, n_bytes = 0;
                for (int c = c_first; c <= c_last; ++c) {
                    const uint32_t mc = (s_cm[c >> 3] >> (4 * (c & 7))) & 15u;
                    if (mc == 0u) continue;                                // no tile of the unit charges this bin
                    const uint32_t bytes = (uint32_t)__popc(mc) * A_BLOCK_BYTES + b_cta;
                    // runs of consecutive charged blocks: {first block, length}, at most two in four bits
                    const int r0b = __ffs(mc) - 1, r0n = __ffs(~(mc >> r0b)) - 1;
                    const int rest = mc & ~(((1 << r0n) - 1) << r0b);
                    const int r1b = rest ? __ffs(rest) - 1 : 0, r1n = rest ? __popc(rest) : 0;
                    const uint32_t st = base + s * stage_sz, fb = full0 + 8 * s;
                    RTC_T(p0);
                    mbar_wait(empty0 + 8 * s, ph ^ 1u);
                    RTC_T(p1);
                    hdr[s].x = u;  hdr[s].y = d;  hdr[s].z = c | ((int)mc << 16) | (mask << 20);
                    hdr[s].w = (c == c_first ? HDR_FIRST : 0) | (c == c_last ? HDR_LAST : 0);
                    mbar_expect_tx(fb, bytes);                         // release: the header is visible to the waiter
                    const unsigned char *Ac = Ab + (size_t)c * NBLK * A_BLOCK_BYTES;
                    // the blocks of a stage sit back to back in charged-block order, whatever their number
                    bulk_g2s(st, Ac + r0b * A_BLOCK_BYTES, (uint32_t)r0n * A_BLOCK_BYTES, fb);
                    if (r1n) bulk_g2s(st + r0n * A_BLOCK_BYTES, Ac + r1b * A_BLOCK_BYTES, (uint32_t)r1n * A_BLOCK_BYTES, fb);
                    bulk_g2s(st + a_area, Bd + (size_t)c * b_stride, b_cta, fb);
                    RTC_T(p2);  RTC_ADD(8, p1 - p0);  RTC_ADD(9, p2 - p1);  RTC_ADD(10, 1);
                    n_mma += 2ull * (unsigned long long)__popc(mc);
                    n_bytes += bytes;
                    if (++s == S) { s = 0; ph ^= 1u; }
                }
                if (leader) {                                          // per item: 2 MMAs per charged (bin, block), bytes of the unit
                    atomicAdd(a.stats + 1, n_mma);
                    atomicAdd(a.stats + 2, n_bytes * (CTA2 ? 2ull : 1ull));
                    atomicAdd(a.stats + 5, 1ull);
                }
                q = q_next;
            }
            mbar_wait(empty0 + 8 * s, ph ^ 1u);                        // terminator: a header-only stage
            hdr[s].w = HDR_END;
            mbar_arrive(full0 + 8 * s);
            RTC_FLUSH;
        }
    } else if (warp == 1 || warp == 6) {
        if (lane == 0 && !leader && warp == 1) {
            // ---------------------------------------------------------------------- relay (peer): this CTA's share of
            // stage s has landed -> tell the leader's MMA issuer.  Nothing but the barrier needs ordering here: what it
            // reports was written by the async proxy (TMA) and is read by the async proxy (tensor core).
            const uint32_t lead_pfull0 = mapa(pfull0, 0u);
            int s = 0;
            uint32_t ph = 0;
            while (true) {
                mbar_wait(full0 + 8 * s, ph);
                const int flags = hdr[s].w;
                mbar_arrive_remote_relaxed(lead_pfull0 + 8 * s);
                if (flags & HDR_END) break;
                if (++s == S) { s = 0; ph ^= 1u; }
            }
        }
        if (lane == 0 && leader) {
            // ---------------------------------------------------------------------- MMA issuers (leader): warp 1 takes the
            // even 16-tick blocks (first accumulator) and hands the items to the epilogue, warp 6 the odd blocks (second
            // accumulator).  One thread issues a tcgen05.mma every ~90 cycles at best, below the 118 cycles the tensor
            // core needs for one, and pays ~400 cycles per stage for its waits, header and commit on top (measured):
            // a single issuer cannot keep the pipe busy.  The two accumulators are independent, so the order between
            // the two threads' MMAs does not matter; each commits every stage (and item) once.
            const int par = warp == 1 ? 0 : 1;
            RTC_DECL;
            // instruction descriptor: D fp32, A and B fp16 (kind::f16) or e4m3 (kind::f8f6f4) -- format code 0 in both
            // kinds --, both K-major, N = NBW, M = 128 per CTA
            const uint32_t idesc = (1u << 4) | ((uint32_t)(NBW >> 3) << 17) | ((uint32_t)((CTA2 ? 2 * TB : TB) >> 4) << 24);
            const uint32_t peer_epi = CTA2 ? mapa(epi0, 1u) : 0u, peer_titem = CTA2 ? mapa(titem, 1u) : 0u;
            int s = 0;
            uint32_t ph = 0, tph = 0;
            while (true) {
                RTC_T(t0);
                mbar_wait(full0 + 8 * s, ph);
                RTC_T(t1);
                if (CTA2) mbar_wait(pfull0 + 8 * s, ph);
                RTC_T(t2);
                int u, d, cz, flags;
                asm volatile("ld.volatile.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(u), "=r"(d), "=r"(cz), "=r"(flags) : "r"(hdr0 + 16 * s) : "memory");
                const int mask = (cz >> 16) & 15, umask = (cz >> 20) & 15;
                if (flags & HDR_END) {
                    if (par) break;
                    mbar_wait_cluster(tempty, tph);                    // the epilogues have read the previous item slot
                    epi_item->w = HDR_END;
                    mbar_arrive(titem);
                    if (CTA2) { st_cluster_v4(peer_epi, 0, 0, 0, HDR_END);  mbar_arrive_remote(peer_titem); }
                    break;
                }
                if (flags & HDR_FIRST) {
                    RTC_T(w0);
                    mbar_wait_cluster(tempty, tph);                    // accumulators drained and zeroed, in both CTAs
                    RTC_T(w1);  RTC_ADD(6, w1 - w0);  RTC_ADD(7, 1);
                    tph ^= 1u;
                    if (!par) {
                        epi_item->x = u;  epi_item->y = d;  epi_item->z = umask;  epi_item->w = 0;
                        mbar_arrive(titem);                            // release: hands the item to the epilogue
                        if (CTA2) { st_cluster_v4(peer_epi, u, d, umask, 0);  mbar_arrive_remote(peer_titem); }
                    }
                }
                tc_fence_after();
                RTC_T(t3);
                const uint32_t st = base + s * stage_sz;
                const uint64_t bd16 = smem_desc(st + a_area, 128, 256, 0), bd8 = smem_desc(st + a_area + b_cta / 2, 128, 256, 0);
                uint32_t src = st;
#pragma unroll
                for (int b = 0; b < NBLK; ++b) {
                    if (!(mask >> b & 1)) continue;                    // no tile of the unit has charge in these 16 ticks
                    if ((b & 1) == par) {
                        const uint32_t dcol = tmem + (b & 1 ? ACC_COL : 0) + 32 * (b >> 1);
                        tc_mma<CTA2>(false, dcol, smem_desc(src, 16, 256, A_LAYOUT), bd16, idesc);
                        tc_mma<CTA2>(true, dcol, smem_desc(src + A_PART_BYTES, 16, 256, A_LAYOUT), bd8, idesc);
                    }
                    src += A_BLOCK_BYTES;
                }
                RTC_T(t4);
                tc_commit_x<CTA2>(empty0 + 8 * s, true);               // stage free, in both CTAs, once these MMAs have read it
                if (flags & HDR_LAST) tc_commit_x<CTA2>(tfull, true);  // accumulators complete, in both CTAs
                RTC_T(t5);
                RTC_ADD(0, t1 - t0);  RTC_ADD(1, t2 - t1);  RTC_ADD(2, t3 - t2);  RTC_ADD(3, t4 - t3);  RTC_ADD(4, t5 - t4);  RTC_ADD(5, 1);
                if (++s == S) { s = 0; ph ^= 1u; }
            }
            RTC_FLUSH;
        }
    } else {
        // ---------------------------------------------------------------------- epilogue (warps 2-5, every CTA)
        const int quad = warp & 3;                                     // TMEM lanes [32 quad, 32 quad + 32)
        const int grp = warp < 6 ? 0 : 1 + (warp - 7) / 4;             // which of the quarter's EPI_G warps
        const uint32_t tlane = tmem + ((uint32_t)(32 * quad) << 16);
        const uint32_t lead_tempty = CTA2 ? mapa(tempty, 0u) : tempty;
        // column chunks of 16 output ticks: group grp reads chunks [ch_lo, ch_hi)
        const int n_ch = (a.tile_ticks + 15) / 16, ch_per = (n_ch + EPI_G - 1) / EPI_G;
        const int ch_lo = min(grp * ch_per, n_ch), ch_hi = min(ch_lo + ch_per, n_ch);
        // every MMA accumulates: the accumulators are zero before the first item and zeroed again after each read-out
        // (each group the 64-column blocks c0 / 64 = grp mod EPI_G, once all groups of the quarter have read)
        for (int c0 = 64 * grp; c0 < 512; c0 += 64 * EPI_G) tmem_zero64(tlane + c0);
        asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        tc_fence_before();
        __syncwarp();
        if (lane == 0) { if (CTA2) mbar_arrive_remote(lead_tempty); else mbar_arrive(tempty); }
        uint32_t iph = 0;
        RTC_DECL;
        while (true) {
            // one lane polls (128 threads spinning on a barrier for the ~30 us an item takes cost issue slots and power)
            if (lane == 0) mbar_wait_cluster(titem, iph);              // acquire: the MMA warp has published the item
            __syncwarp();
            if (epi_item->w & HDR_END) break;
            const int u = epi_item->x, d = epi_item->y, mask = epi_item->z;
            // (the tile's scale and block counts come from HBM / L2: fetched while the item's MMAs still run)
            const int tile = (u * (CTA2 ? 2 : 1) + (int)rank) * TB + 32 * quad + lane;
            const bool live = tile < a.n_tiles;
            const bool even = (mask & 5) != 0, odd = (mask & 10) != 0;
            float scale = 0.f;
            float nzb[NBLK] = {0.f, 0.f, 0.f, 0.f};
            if (live) {
                const int4 tm = *(const int4 *)(a.tile_meta + 4 * tile);
                scale = __int_as_float((127 + tm.z - a.b_scale_log2) << 23);
#pragma unroll
                for (int b = 0; b < NBLK; ++b) nzb[b] = (float)(((unsigned)tm.w >> (8 * b)) & 255u) * (8.f / 16.f) * a.kappa;
            }
            if (lane == 0) mbar_wait(tfull, iph);
            __syncwarp();
            tc_fence_after();
            RTC_T(e0);
            // 1 + kappa x (non-zero cells with arrival tick j in (n - K, n], of the blocks of one parity): what the
            // accumulator column of output tick n lost to truncation, in expectation.  Cells are taken as spread evenly
            // over the 16 ticks of their block; evaluated every 8 ticks, linear in between.
            auto comp = [&](int n, int par) -> float {
                const int m = n - a.K;
                const int wa = min(max(n - 16 * par + 1, 0), 16) - min(max(m - 16 * par + 1, 0), 16);
                const int wb = min(max(n - 16 * par - 31, 0), 16) - min(max(m - 16 * par - 31, 0), 16);
                return fmaf(nzb[par], (float)wa, fmaf(nzb[par + 2], (float)wb, 1.f));
            };
            float *dst = a.partial + ((size_t)(live ? tile : 0) * a.WW + d) * a.tile_ticks;
            float g0e = comp(16 * ch_lo, 0), g0o = comp(16 * ch_lo, 1);
            // output tick n = even accumulator column n (blocks 0, 2) + odd accumulator column n - 16 (blocks 1, 3)
            for (int n0 = 16 * ch_lo; n0 < 16 * ch_hi; n0 += 16) {
                uint32_t v0[16], v1[16];
                const bool has0 = even && n0 < ACC_COL, has1 = odd && n0 >= 16;
                if (has0) tmem_ld16(tlane + n0, v0);
                if (has1) tmem_ld16(tlane + ACC_COL + n0 - 16, v1);
                const float g1e = comp(n0 + 8, 0), g1o = comp(n0 + 8, 1), g2e = comp(n0 + 16, 0), g2o = comp(n0 + 16, 1);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                if (live) {
                    const int nv = min(16, a.tile_ticks - n0);         // tile_ticks is a multiple of 8
#pragma unroll
                    for (int i8 = 0; i8 < 2; ++i8) {                   // 8 ticks = one 32-byte sector of the row per store
                        if (8 * i8 >= nv) break;
                        const float be = (i8 == 0 ? g0e : g1e) * scale, bo = (i8 == 0 ? g0o : g1o) * scale;   // value at the 8-tick node
                        const float se = (i8 == 0 ? g1e - g0e : g2e - g1e) * (0.125f * scale), so = (i8 == 0 ? g1o - g0o : g2o - g1o) * (0.125f * scale);
                        float r[8];
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const float t = (float)k;
                            const float x0 = has0 ? __uint_as_float(v0[8 * i8 + k]) : 0.f, x1 = has1 ? __uint_as_float(v1[8 * i8 + k]) : 0.f;
                            r[k] = fmaf(x0, fmaf(se, t, be), x1 * fmaf(so, t, bo));
                        }
                        // one 256-bit store per 8 ticks: each lane writes its own row, so the store path sees 32 sectors per
                        // instruction either way, and half as many instructions (response 175 -> 167 ms at configs[3])
                        st_global_256(dst + n0 + 8 * i8, make_uint4(__float_as_uint(r[0]), __float_as_uint(r[1]), __float_as_uint(r[2]), __float_as_uint(r[3])),
                                      make_uint4(__float_as_uint(r[4]), __float_as_uint(r[5]), __float_as_uint(r[6]), __float_as_uint(r[7])));
                    }
                }
                g0e = g2e;  g0o = g2o;
            }
            RTC_T(eA);
            if (EPI_G > 1) {                                           // the quarter's columns are read by all its groups
                tc_fence_before();
                asm volatile("bar.sync %0, %1;" ::"r"(1 + quad), "r"(32 * EPI_G) : "memory");
                tc_fence_after();
            }
            for (int c0 = 64 * grp; c0 < 2 * ACC_COL; c0 += 64 * EPI_G)
                if (c0 < ACC_COL ? even : odd) tmem_zero64(tlane + c0);
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            RTC_T(eB);
            tc_fence_before();
            __syncwarp();
            if (lane == 0) { if (CTA2) mbar_arrive_remote(lead_tempty); else mbar_arrive(tempty); }
            iph ^= 1u;
            RTC_T(e1);
            if (tid == 64) { RTC_ADD(11, e1 - e0);  RTC_ADD(12, 1);  RTC_ADD(13, eA - e0);  RTC_ADD(14, eB - eA); }
        }
        if (tid == 64) RTC_FLUSH;
    }
    tc_fence_before();
    __syncthreads();
    if (CTA2) cluster_sync_all();                                      // nobody leaves while its partner may still signal it
    if (warp == 1) {
        tc_fence_after();
        if (CTA2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
        else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    }
}

}  // namespace rtc
