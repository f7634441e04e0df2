// Tensor-pipe contraction step for sm_100a: a pairwise contraction whose outer dimensions are large is a
// batched GEMM (section 3.2; cost dim(i) dim(j) dim(k), lines 407-412)
//     C_r[outA(i) | outB(j)] = sum_k A_r[i, k] * B_r[j, k],   M = 4^{#outer_lhs}, N = 4^{#outer_rhs}, K = 4^{#inner}
// per state r.  Both operands are K-major fp32 in HBM/L2.  tcgen05 has no fp32-input MMA, so each operand
// tile is split in shared memory into a_hi (top 19 bits, exactly a TF32 value) and a_lo = a - a_hi (exact in fp32)
// and three TF32 MMAs hi*hi + hi*lo + lo*hi accumulate in fp32 in TMEM.
//
// Persistent, warp-specialised CTA (one per SM), 384 threads:
//   warp 0      TMA producer: cp.async.bulk.tensor 3-D tiles {32 k, 128 or BN rows, 1 state} with 128-byte swizzle;
//               the state coordinate of a LEAF/TABLE operand is the state's key (a3 gather = a TMA coordinate)
//   warp 1      MMA issuer: one elected lane, 12 tcgen05.mma.kind::tf32 per k-block, tcgen05.commit frees the stage
//   warps 2-9   accumulate + epilogue: tcgen05.ld -> fp32 round-to-nearest adds in registers -> scatter to C; BN = 128: two
//               groups of four warps (one per TMEM lane quadrant), each owning half of the tile's columns; BN <= 64: warps 2-5
//   warps 6-9   BN <= 64 only: A splitter - a thread per tile row reads the landed raw row once, splits it in registers and
//               writes hi and lo into TENSOR MEMORY (tcgen05.st), the MMAs take A from there (tcgen05.mma with a TMEM A operand)
//   warps 10-11 splitter: fp32 tile -> hi (in place) and lo (second buffer), same swizzled byte offsets (BN <= 64: B only)
// Pipelines: full[s] (TMA -> splitters), ready[s] (splitters -> MMA), empty[s] (MMA -> TMA, and -> A splitter: the TMEM A
// buffer of k-block it - 2 is free).
// The tensor pipe's fp32 accumulator rounds toward zero on every add (measured: -5e-8 relative per accumulation,
// profiles/r01c notes), a bias that grows with the number of k-steps.  So (i) the hi*hi products of at most
// TC_CHUNK_KB k-blocks (8 MMAs) accumulate in a TMEM buffer D_hi that the accumulate warps then drain and add to
// registers in round-to-nearest, two D_hi buffers alternating so draining overlaps the next chunk's MMAs; (ii) the
// hi*lo + lo*hi products, 2^-11 smaller, accumulate over the whole K in their own buffer D_lo (two of them,
// alternating per tile), where the same bias is negligible.  TMEM columns: 4 x BN <= 512 (BN <= 64: + 2 x 64 for A).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "device_args.h"

namespace tqc {

constexpr int TC_BM = 128;          // UMMA M
constexpr int TC_BK = 32;           // fp32 elements per k-block = 128 bytes = one swizzle row
constexpr int TC_THREADS = 384;      // 12 warps: TMA, MMA, 2 x 4 accumulate/epilogue warps, 2 splitter warps
constexpr int TC_SPLIT_THREADS = 64;
constexpr int TC_CHUNK_KB = 1;       // k-blocks (of 32) whose hi*hi products accumulate in TMEM before a drain (4 accumulations)

struct TcArgs {
    const uint32_t *keysA, *keysB;  // state coordinate of a keyed operand (null: the row itself)
    float *C;
    long long c_row_stride;
    BitMap outA, outB;              // i -> C offset bits, j -> C offset bits
    int lgM, lgN, lgK;
    int R;                          // states in this launch
    int BN;                         // N tile: 16, 32, 64 or 128
    int stages;
    int mask_hi;                    // hi = TF32 value nearest to x, written back in place (else: x itself, truncated by the MMA)
    int vec4;                       // 4 consecutive j are contiguous in C (pair kernel: 1 = j, j+1 adjacent; 2 = j .. j+3)
    int chunk_kb;                   // k-blocks per hi*hi drain (0: TC_CHUNK_KB)
    unsigned long long *trace;      // develop builds: clock64 stamps of the first k-blocks of cluster 0 (kernels_tc2.cuh)
    int debug;                      // development knobs (TQC_TC_DEBUG): 1 no global stores, 2 no store phase, 4 no split, 8 no drains
};

// development knobs (TcArgs.debug) exist only in -DTQC_DEVELOP builds; a release build compiles every test of them away
#ifdef TQC_DEVELOP
#define TQC_DBG(a, bit) (((a).debug & (bit)) != 0)
#else
#define TQC_DBG(a, bit) false
#endif

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

__device__ __forceinline__ void tma_load_3d(const CUtensorMap *map, uint64_t *bar, void *dst, int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

// K-major, 128-byte-swizzled operand tile: rows of 128 bytes, 8-row groups 1024 bytes apart.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);          // start address, 16-byte units
    d |= (uint64_t)1 << 16;                                // leading byte offset (unused for swizzled K-major)
    d |= (uint64_t)(1024 >> 4) << 32;                      // stride byte offset between 8-row groups
    d |= (uint64_t)1 << 46;                                // descriptor version (sm_100)
    d |= (uint64_t)2 << 61;                                // SWIZZLE_128B
    return d;
}

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
// A operand from TENSOR MEMORY (lane = row, one 32-bit column per K element), B from a shared-memory descriptor
__device__ __forceinline__ void umma_tf32_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "r"(tmem_a), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
// 16 consecutive columns of this lane's row
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]),
          "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]),
          "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]),
          "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[32]) {      // 16 columns into v[0..15]
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}


// bit map applied to a small index (a lane id or a column within a vector): same as bitmap_apply
__device__ __forceinline__ unsigned long long bitmap_apply_small(const BitMap &m, unsigned x) { return bitmap_apply(m, (unsigned long long)x); }

template <int NV>
__device__ __forceinline__ void split_tile(uint32_t addr, uint32_t lo_ofs, bool mask_hi) {
    uint4 x[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x[v].x), "=r"(x[v].y), "=r"(x[v].z), "=r"(x[v].w)
                     : "r"(addr + (uint32_t)v * (TC_SPLIT_THREADS * 16u)));
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const uint32_t p = addr + (uint32_t)v * (TC_SPLIT_THREADS * 16u);
        // mask_hi: hi = the TF32 value NEAREST to x (written back in place), so lo = x - hi is signed with zero mean and
        // neither the dropped lo*lo term nor the truncation of lo inside the MMA biases the sum; otherwise hi = x truncated
        const uint32_t rnd = mask_hi ? 0x1000u : 0u;
        const uint4 h = make_uint4((x[v].x + rnd) & 0xFFFFE000u, (x[v].y + rnd) & 0xFFFFE000u, (x[v].z + rnd) & 0xFFFFE000u, (x[v].w + rnd) & 0xFFFFE000u);
        const float l0 = __uint_as_float(x[v].x) - __uint_as_float(h.x), l1 = __uint_as_float(x[v].y) - __uint_as_float(h.y);
        const float l2 = __uint_as_float(x[v].z) - __uint_as_float(h.z), l3 = __uint_as_float(x[v].w) - __uint_as_float(h.w);
        asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(p + lo_ofs), "f"(l0), "f"(l1), "f"(l2), "f"(l3) : "memory");
        if (mask_hi) asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(p), "r"(h.x), "r"(h.y), "r"(h.z), "r"(h.w) : "memory");
    }
}

// float index of element (row i5, column j5) of a warp's staging block: rows of CB floats (32-float pitch for CB = 32,
// 16-float pitch otherwise), float4 slot XOR-swizzled by the row so that row-wise float4 writes and the permuted float4
// reads of the store phase are bank-conflict free
template <int CB>
__device__ __forceinline__ uint32_t scratch_index(uint32_t i5, uint32_t j5) {
    if (CB == 32) {
        const uint32_t rev = ((i5 & 1u) << 2) | (i5 & 2u) | ((i5 >> 2) & 1u);
        return i5 * 32u + ((((j5 >> 2) ^ rev) & 7u) << 2) + (j5 & 3u);
    }
    return i5 * 16u + ((((j5 >> 2) ^ (i5 >> 1)) & 3u) << 2) + (j5 & 3u);
}

template <int BN>
__global__ void __launch_bounds__(TC_THREADS, 1)
step_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const TcArgs a) {
    extern __shared__ unsigned char tc_smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[4], ready_bar[4], empty_bar[4];
    __shared__ __align__(8) uint64_t hi_full_bar[2], hi_empty_bar[2], lo_full_bar[2], lo_empty_bar[2];
    __shared__ uint32_t tmem_base_slot;
    // epilogue: each warp stages 32 rows x CB columns in its own scratch and writes them out in ascending C-offset
    // order (perm tables), so a warp store covers the longest contiguous run the consumer's digit layout allows
    // Narrow tiles (BN <= 64) take the A operand of every MMA from TENSOR MEMORY: a k-block's A tile is read three times by the
    // MMAs (hi twice, lo once) on top of the TMA write and the split, 112 KB of shared-memory traffic per k-block whatever BN,
    // and the narrow steps ran at 0.7-0.8 of that shared-memory floor (measured: 1750 cycles per k-block for BN = 16 ... 64,
    // operand in HBM or in L2 alike).  Warps 6-9 (one per TMEM lane quadrant, a thread per row) read the landed raw rows once,
    // split them in registers and write hi and lo with tcgen05.st into one of two 64-column A buffers; the MMAs are the
    // TMEM-A form.  The accumulate warps are one column group then (warps 2-5), B is split in shared memory as before.
    constexpr bool A_TMEM = BN <= 64;
    constexpr int EG = BN >= 128 ? 2 : 1;            // epilogue warp groups
    constexpr int EC = BN / EG;                       // columns each epilogue warp accumulates
    constexpr int CB = EG == 2 ? 16 : (BN < 32 ? BN : 32);   // columns per staged block
    constexpr int LB = CB == 32 ? 5 : 4;
    // C-offset tables (bit maps applied once per kernel, not per tile): m-tile, lane quadrant, n-tile, column block
    __shared__ uint32_t oa_mt[256], oa_q[4], ob_nt[256], ob_blk[BN / CB];
    __shared__ uint32_t perm_off[32 * CB];
    __shared__ __align__(8) uint16_t perm_src[32 * CB];
    __shared__ __align__(16) float scratch[4 * EG][32 * (CB == 32 ? 32 : 16)];   // row i5: CB/4 float4 slots, XOR-swizzled by the row

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int S = a.stages;
    constexpr uint32_t bytesA = TC_BM * TC_BK * 4, bytesB = (uint32_t)BN * TC_BK * 4;
    constexpr uint32_t stage_bytes = 2 * bytesA + 2 * bytesB;
    unsigned char *tiles = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(tc_smem_raw) + 1023) & ~(uintptr_t)1023);
    auto A_raw = [&](int s) { return tiles + (size_t)s * stage_bytes; };
    auto A_lo = [&](int s) { return tiles + (size_t)s * stage_bytes + bytesA; };
    auto B_raw = [&](int s) { return tiles + (size_t)s * stage_bytes + 2 * bytesA; };
    auto B_lo = [&](int s) { return tiles + (size_t)s * stage_bytes + 2 * bytesA + bytesB; };

    const int n_kb = 1 << (a.lgK - 5);
    const int chunk_want = a.chunk_kb > 0 ? a.chunk_kb : TC_CHUNK_KB;
    const int chunk_kb = n_kb < chunk_want ? n_kb : chunk_want;
    const int n_chunks = n_kb / chunk_kb;
    const long long tiles_m = 1ll << (a.lgM - 7);
    const long long tiles_n = (1ll << a.lgN) / BN;
    const long long total = tiles_m * tiles_n * a.R;
    // D_hi[0], D_hi[1], D_lo[0], D_lo[1]; with A_TMEM two A buffers of 64 columns (hi 32, lo 32) behind them
    constexpr uint32_t tmem_cols = !A_TMEM ? (uint32_t)(4 * BN) : (4 * BN + 128 <= 256 ? 256u : 512u);

    // ---- one-time setup -------------------------------------------------------------------------
    for (int x = threadIdx.x; x < 256; x += TC_THREADS) {
        oa_mt[x] = x < tiles_m ? (uint32_t)bitmap_apply(a.outA, (unsigned long long)x * TC_BM) : 0u;
        ob_nt[x] = x < tiles_n ? (uint32_t)bitmap_apply(a.outB, (unsigned long long)x * BN) : 0u;
        if (x < 4) oa_q[x] = (uint32_t)bitmap_apply(a.outA, (unsigned long long)x * 32);
        if (x < BN / CB) ob_blk[x] = (uint32_t)bitmap_apply(a.outB, (unsigned long long)x * CB);
    }
    for (int e = threadIdx.x; e < 32 * CB; e += TC_THREADS) {
        // the 5 + LB index bits of a block, ordered by the C-offset bit they map to
        uint32_t dst[5 + LB], src[5 + LB];
#pragma unroll
        for (int b = 0; b < 5 + LB; ++b) {
            const unsigned long long o = b < 5 ? bitmap_apply(a.outA, 1ull << b) : bitmap_apply(a.outB, 1ull << (b - 5));
            dst[b] = (uint32_t)(__ffsll((long long)o) - 1);
            src[b] = (uint32_t)b;
        }
#pragma unroll
        for (int x = 1; x < 5 + LB; ++x)                     // insertion sort by destination bit
#pragma unroll
            for (int y = x; y > 0; --y)
                if (dst[y] < dst[y - 1]) { uint32_t t0 = dst[y]; dst[y] = dst[y - 1]; dst[y - 1] = t0; t0 = src[y]; src[y] = src[y - 1]; src[y - 1] = t0; }
        uint32_t off = 0, ij = 0;
#pragma unroll
        for (int k = 0; k < 5 + LB; ++k)
            if ((e >> k) & 1) { off |= 1u << dst[k]; ij |= 1u << src[k]; }
        perm_off[e] = off;
        {
            const uint32_t i5 = ij & 31u, j5 = ij >> 5;
            perm_src[e] = (uint16_t)scratch_index<CB>(i5, j5);
        }
    }
    if (threadIdx.x == 0) {
        for (int s = 0; s < S; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&ready_bar[s], TC_SPLIT_THREADS / 32 + (A_TMEM ? 4 : 0)); mbar_init(&empty_bar[s], 1); }
        for (int s = 0; s < 2; ++s) {
            mbar_init(&hi_full_bar[s], 1); mbar_init(&hi_empty_bar[s], 4 * EG);
            mbar_init(&lo_full_bar[s], 1); mbar_init(&lo_empty_bar[s], 4 * EG);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapB) : "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_slot)), "r"(tmem_cols) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = tmem_base_slot;

    if (warp == 0) {
        // ===== TMA producer =====
        if (lane == 0) {
            long long it = 0;
            for (long long t = blockIdx.x; t < total; t += gridDim.x) {
                const long long nt = t % tiles_n, mt = (t / tiles_n) % tiles_m, r = t / (tiles_n * tiles_m);
                const int rowA = a.keysA ? (int)a.keysA[r] : (int)r;
                const int rowB = a.keysB ? (int)a.keysB[r] : (int)r;
                for (int kb = 0; kb < n_kb; ++kb, ++it) {
                    const int s = (int)(it % S);
                    const uint32_t ph = (uint32_t)((it / S) & 1);
                    mbar_wait(&empty_bar[s], ph ^ 1u);
                    if (TQC_DBG(a, 16)) { mbar_arrive(&full_bar[s]); continue; }
                    mbar_expect_tx(&full_bar[s], bytesA + bytesB);
                    tma_load_3d(&mapA, &full_bar[s], A_raw(s), kb * TC_BK, (int)(mt * TC_BM), rowA);
                    tma_load_3d(&mapB, &full_bar[s], B_raw(s), kb * TC_BK, (int)(nt * BN), rowB);
                }
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer =====
        constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(TC_BM >> 4) << 24);
        long long it = 0, lt = 0, g = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x, ++lt) {
            const uint32_t lb = (uint32_t)(lt & 1), lph = (uint32_t)((lt >> 1) & 1);
            mbar_wait(&lo_empty_bar[lb], lph ^ 1u);
            const uint32_t d_lo = tmem_base + (2u + lb) * (uint32_t)BN;
            int kb = 0;
            for (int c = 0; c < n_chunks; ++c, ++g) {
                const uint32_t hb = (uint32_t)(g & 1), hph = (uint32_t)((g >> 1) & 1);
                mbar_wait(&hi_empty_bar[hb], hph ^ 1u);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d_hi = tmem_base + hb * (uint32_t)BN;
                for (int kc = 0; kc < chunk_kb; ++kc, ++kb, ++it) {
                    const int s = (int)(it % S);
                    const uint32_t ph = (uint32_t)((it / S) & 1);
                    // hi*hi reads only the raw tiles (TMA wrote them: no proxy fence needed), so it starts as soon as the
                    // load lands and overlaps the splitter; the lo terms wait for the splitter's ready barrier
                    // (with round-to-nearest hi parts the raw tiles are rewritten by the splitter: wait for it first)
                    mbar_wait((a.mask_hi || A_TMEM) ? &ready_bar[s] : &full_bar[s], ph);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    const uint64_t dah = umma_desc_sw128(smem_u32(A_raw(s))), dal = umma_desc_sw128(smem_u32(A_lo(s)));
                    const uint64_t dbh = umma_desc_sw128(smem_u32(B_raw(s))), dbl = umma_desc_sw128(smem_u32(B_lo(s)));
                    const bool run = !TQC_DBG(a, 32) || (kb | kc) == 0;
                    if constexpr (A_TMEM) {
                        // ready = A hi / lo of this k-block in TMEM buffer it & 1 and B split in shared memory
                        const uint32_t a_hi = tmem_base + 4u * (uint32_t)BN + 64u * (uint32_t)(it & 1), a_lo = a_hi + 32u;
                        if (lane == 0) {
                            if (run) {
#pragma unroll
                                for (int k = 0; k < TC_BK / 8; ++k) {
                                    const uint64_t adv = (uint64_t)(k * 8 * 4 >> 4);
                                    umma_tf32_ts(d_lo, a_lo + 8u * k, dbh + adv, idesc, (kb | k) ? 1u : 0u);
                                    umma_tf32_ts(d_lo, a_hi + 8u * k, dbl + adv, idesc, 1u);
                                }
#pragma unroll
                                for (int k = 0; k < TC_BK / 8; ++k) {
                                    const uint64_t adv = (uint64_t)(k * 8 * 4 >> 4);
                                    umma_tf32_ts(d_hi, a_hi + 8u * k, dbh + adv, idesc, (kc | k) ? 1u : 0u);
                                }
                            }
                            umma_commit(&empty_bar[s]);
                            if (kc == chunk_kb - 1) umma_commit(&hi_full_bar[hb]);
                            if (kb == n_kb - 1) umma_commit(&lo_full_bar[lb]);
                        }
                        __syncwarp();
                        continue;
                    }
                    if (lane == 0 && run) {
#pragma unroll
                        for (int k = 0; k < TC_BK / 8; ++k) {
                            const uint64_t adv = (uint64_t)(k * 8 * 4 >> 4);       // 32 bytes per K=8 slice, 16-byte units
                            umma_tf32(d_hi, dah + adv, dbh + adv, idesc, (kc | k) ? 1u : 0u);
                        }
                    }
                    __syncwarp();
                    mbar_wait(&ready_bar[s], ph);
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    if (lane == 0) {
                        if (run) {
#pragma unroll
                            for (int k = 0; k < TC_BK / 8; ++k) {
                                const uint64_t adv = (uint64_t)(k * 8 * 4 >> 4);
                                umma_tf32(d_lo, dal + adv, dbh + adv, idesc, (kb | k) ? 1u : 0u);
                                umma_tf32(d_lo, dah + adv, dbl + adv, idesc, 1u);
                            }
                        }
                        umma_commit(&empty_bar[s]);                                 // frees the stage when these MMAs retire
                        if (kc == chunk_kb - 1) umma_commit(&hi_full_bar[hb]);
                        if (kb == n_kb - 1) umma_commit(&lo_full_bar[lb]);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp < 2 + 4 * EG) {
        // ===== accumulate (round-to-nearest, registers) + epilogue =====
        const int w4 = warp & 3;
        const int col_base = ((warp - 2) >> 2) * EC;             // this warp's first column of the tile
        const uint32_t lane_base = (uint32_t)(32 * w4) << 16;
        uint32_t rd_ofs[CB / 4], st_ofs[CB / 4];           // this lane's float4 slots of a block, in ascending C-offset order
#pragma unroll
        for (int p = 0; p < CB / 4; ++p) { rd_ofs[p] = perm_src[(p * 32 + lane) * 4]; st_ofs[p] = perm_off[(p * 32 + lane) * 4]; }
        long long lt = 0, g = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x, ++lt) {
            const long long nt = t % tiles_n, mt = (t / tiles_n) % tiles_m, r = t / (tiles_n * tiles_m);
            float acc[EC];
#pragma unroll
            for (int q = 0; q < EC; ++q) acc[q] = 0.f;
            for (int c = 0; c < n_chunks; ++c, ++g) {
                const uint32_t hb = (uint32_t)(g & 1), hph = (uint32_t)((g >> 1) & 1);
                mbar_wait(&hi_full_bar[hb], hph);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t taddr = tmem_base + lane_base + hb * (uint32_t)BN + (uint32_t)col_base;
                if (!TQC_DBG(a, 8))
#pragma unroll
                for (int c0 = 0; c0 < EC; c0 += 32) {
                    uint32_t v[32];
                    if (EC - c0 >= 32) tmem_ld32(taddr + c0, v); else tmem_ld16(taddr + c0, v);
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                    for (int q = 0; q < 32; ++q)
                        if (c0 + q < EC) acc[c0 + q] += __uint_as_float(v[q]);
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                __syncwarp();
                if (lane == 0) mbar_arrive(&hi_empty_bar[hb]);
            }
            const uint32_t lb = (uint32_t)(lt & 1), lph = (uint32_t)((lt >> 1) & 1);
            mbar_wait(&lo_full_bar[lb], lph);
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            float *crow = a.C + r * a.c_row_stride + (oa_mt[mt] | oa_q[w4] | ob_nt[nt]);
            const uint32_t laddr = tmem_base + lane_base + (2u + lb) * (uint32_t)BN + (uint32_t)col_base;
#pragma unroll
            for (int c0 = 0; c0 < EC; c0 += 32) {
                uint32_t v[32];
                if (EC - c0 >= 32) tmem_ld32(laddr + c0, v); else tmem_ld16(laddr + c0, v);
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int q = 0; q < 32; ++q)
                    if (c0 + q < EC) acc[c0 + q] += __uint_as_float(v[q]);
            }
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&lo_empty_bar[lb]);
            float *scr = scratch[warp - 2];
            if (TQC_DBG(a, 2)) continue;
#pragma unroll
            for (int c0 = 0; c0 < EC; c0 += CB) {
                __syncwarp();
#pragma unroll
                for (int k = 0; k < CB / 4; ++k)
                    *reinterpret_cast<float4 *>(scr + scratch_index<CB>((uint32_t)lane, (uint32_t)(4 * k))) =
                        make_float4(acc[c0 + 4 * k], acc[c0 + 4 * k + 1], acc[c0 + 4 * k + 2], acc[c0 + 4 * k + 3]);
                __syncwarp();
                float *cblk = crow + ob_blk[(col_base + c0) / CB];
                if (a.vec4) {
#pragma unroll
                    for (int p = 0; p < CB / 4; ++p) {
                        const float4 val = *reinterpret_cast<const float4 *>(scr + rd_ofs[p]);
                        if (!TQC_DBG(a, 1) || val.x == 123.456f) *reinterpret_cast<float4 *>(cblk + st_ofs[p]) = val;
                    }
                } else if (perm_off[1] == 1u && perm_off[2] == 2u && perm_off[3] == 3u) {
                    // four consecutive elements of the ascending order are contiguous in C (the two lowest C bits lie inside
                    // the block) but not in the staging block: four scalar reads, one 16-byte store
#pragma unroll
                    for (int p = 0; p < CB / 4; ++p) {
                        const int e = (p * 32 + lane) * 4;
                        const uint2 ps = *reinterpret_cast<const uint2 *>(perm_src + e);
                        const float4 val = make_float4(scr[ps.x & 0xFFFFu], scr[ps.x >> 16], scr[ps.y & 0xFFFFu], scr[ps.y >> 16]);
                        *reinterpret_cast<float4 *>(cblk + st_ofs[p]) = val;
                    }
                } else {
#pragma unroll
                    for (int p = 0; p < CB; ++p) {
                        const int e = p * 32 + lane;
                        cblk[perm_off[e]] = scr[perm_src[e]];
                    }
                }
            }
        }
    } else if (A_TMEM && warp >= 6 && warp < 10) {
        // ===== A splitter (narrow tiles): raw row -> registers -> hi / lo in tensor memory =====
        const uint32_t row = (uint32_t)(32 * (warp & 3) + lane);          // TMEM lane = tile row; a warp owns its lane quadrant
        const uint32_t lane_base = (uint32_t)(32 * (warp & 3)) << 16;
        const bool mask_hi = a.mask_hi != 0;
        const long long my_kb = ((long long)blockIdx.x < total ? (total - blockIdx.x + gridDim.x - 1) / gridDim.x : 0) * n_kb;
        for (long long it = 0; it < my_kb; ++it) {
            const int s = (int)(it % S);
            if (it >= 2) {                                                // the MMAs that read this A buffer (k-block it - 2) have retired
                const long long jt = it - 2;
                mbar_wait(&empty_bar[(int)(jt % S)], (uint32_t)((jt / S) & 1));
            }
            mbar_wait(&full_bar[s], (uint32_t)((it / S) & 1));
            asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
            const uint32_t src = smem_u32(A_raw(s)) + row * 128u;
            const uint32_t a_hi = tmem_base + lane_base + 4u * (uint32_t)BN + 64u * (uint32_t)(it & 1), a_lo = a_hi + 32u;
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                uint32_t x[16], h[16], l[16];
#pragma unroll
                for (int c = 0; c < 4; ++c) {                             // 16-byte chunk 4 half + c of the row sits at slot chunk ^ (row & 7)
                    const uint32_t chunk = (uint32_t)(4 * half + c);
                    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x[4 * c]), "=r"(x[4 * c + 1]), "=r"(x[4 * c + 2]), "=r"(x[4 * c + 3])
                                 : "r"(src + ((chunk ^ (row & 7u)) << 4)));
                }
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    h[e] = (x[e] + (mask_hi ? 0x1000u : 0u)) & 0xFFFFE000u;
                    l[e] = __float_as_uint(__uint_as_float(x[e]) - __uint_as_float(h[e]));
                }
                tmem_st16(a_hi + 16u * half, h);
                tmem_st16(a_lo + 16u * half, l);
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
            asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(&ready_bar[s]);
        }
    } else if (warp >= (TC_THREADS - TC_SPLIT_THREADS) / 32) {
        // ===== splitter: fp32 -> hi (in place) + lo =====
        const int st = threadIdx.x - (TC_THREADS - TC_SPLIT_THREADS);
        const bool mask_hi = a.mask_hi != 0;
        long long it = 0;
        for (long long t = blockIdx.x; t < total; t += gridDim.x) {
            for (int kb = 0; kb < n_kb; ++kb, ++it) {
                const int s = (int)(it % S);
                const uint32_t ph = (uint32_t)((it / S) & 1);
                mbar_wait(&full_bar[s], ph);
                // per stage: [A_raw][A_lo][B_raw][B_lo]; element e of a raw tile and of its lo tile share the swizzled offset
                const uint32_t sa = smem_u32(A_raw(s)) + (uint32_t)st * 16u;
                if (!TQC_DBG(a, 4) && !A_TMEM)
                split_tile<(int)(bytesA >> 4) / TC_SPLIT_THREADS>(sa, bytesA, mask_hi);
                if (!TQC_DBG(a, 4))
                split_tile<(int)(bytesB >> 4) / TC_SPLIT_THREADS>(sa + 2u * bytesA, bytesB, mask_hi);
                if (!TQC_DBG(a, 64)) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy writes -> visible to the MMA's async proxy
                __syncwarp();
                if (lane == 0) mbar_arrive(&ready_bar[s]);
            }
        }
    }

    // ---- teardown ---------------------------------------------------------------------------------
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(tmem_cols) : "memory");
    }
}

}  // namespace tqc
