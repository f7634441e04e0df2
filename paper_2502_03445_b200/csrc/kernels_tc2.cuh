// Tensor-pipe contraction step on CTA PAIRS (tcgen05 cta_group::2) for sm_100a: the same batched product as kernels_tc.cuh
//     C_r[outA(i) | outB(j)] = sum_k A_r[i, k] * B_r[j, k]          (cost lines 407-412)
// with 256 x BN tiles computed by the two SMs of a cluster.  Why pairs: a kind::tf32 MMA reads 32 bytes of K per operand
// row from shared memory, and with 3xTF32 every k-block is read by twelve MMAs, so the one-CTA kernels are bound by the
// shared-memory port and by L2 -> shared-memory operand traffic (measured, profiles/r02 notes: the 128 x 128 kernel spends
// as long loading, splitting and draining as it would spend on its MMAs).  In a pair each CTA stages only ITS 128 rows of A
// and ITS half of the B tile, both tensor cores read both halves of B, and each CTA accumulates 128 x BN outputs: half
// the operand bytes per flop in L2 traffic, in TMA writes, in splitter traffic and in MMA operand reads.
//
// One CTA = 20 warps:
//   warp 0       TMA producer (one lane): its CTA's A rows and B-half rows of every k-block (32 fp32 = one 128-byte swizzle
//                row), 3-D maps {K, rows, state-or-key} as in kernels_tc.cuh
//   warp 1       MMA issuer, LEADER CTA only (one lane): per k-block 8 lo MMAs then 4 hi*hi MMAs into one of two TMEM
//                accumulators (BN columns each), tcgen05.commit multicast to both CTAs
//   warps 2-3    splitters: the landed stage A -> hi = TF32 nearest (in place) and lo (second tile); B is used as it is for hi
//                (the MMA reads the top 19 bits: a truncation) and gets a lo tile, every lo rounded to TF32 so that what the
//                MMA drops is zero-mean; with the A residual signed and zero-mean the dropped lo*lo term has no bias either
//   warps 4-19   accumulate + store: drain the accumulator of every k-block (tcgen05.ld 16x256b) and add it to registers in
//                round-to-nearest -- the tensor pipe's fp32 accumulator rounds toward zero, so at most the
//                four hi*hi accumulations of one k-block see a full-size sum; then store the finished 32 x BN/4 block straight
//                from registers: in the 16x256b layout a quad of lanes holds 8 consecutive columns of one row, so a warp store
//                writes whole 32-byte sectors whichever operand owns C's lowest digits.
// Splitting (shared-memory port) and draining (TMEM read port) run on different warps because each takes about as long as the
// MMAs of a k-block (measured with the clock64 trace of the develop build: 1500 and 1400 cycles against 1536).
// Barriers: full[s] local (TMA -> splitters); ready[s] in the leader (one arrival per CTA: its splitter warps meet at a named
// barrier first) -> MMA; empty[s] and d_full[b] in both CTAs (multicast commit); d_empty[b] in the leader (one arrival per CTA).
#pragma once
#include "kernels_tc.cuh"

namespace tqc {

constexpr int TC2_DRAIN = 512;            // accumulate / store threads (16 warps after the splitters)
constexpr int TC2_FIRST_SPLIT = 2;        // warp 0 = TMA, warp 1 = MMA, then NSPLIT / 32 splitter warps, then the 16 accumulate warps
// splitter threads: 64 for the 256-column tile (its accumulate warps hold 64 accumulators each and the CTA is at the register
// limit with 20 warps); 128 for narrower tiles, whose k-blocks are shorter while the A tile to split stays the same
__host__ __device__ constexpr int tc2_split_threads(int BN) { return BN >= 256 ? 64 : 128; }      // only BN = 256 is instantiated
__host__ __device__ constexpr int tc2_threads(int BN) { return 64 + tc2_split_threads(BN) + TC2_DRAIN; }
constexpr int TC2_BM = 256;               // pair tile rows (128 per CTA)

__device__ __forceinline__ uint32_t cluster_ctarank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the barrier at the same shared-memory offset in CTA `cta` of the cluster
__device__ __forceinline__ void mbar_arrive_cluster(uint64_t *bar, uint32_t cta) {
    asm volatile(
        "{\n\t"
        ".reg .b32 ra;\n\t"
        "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
        "mbarrier.arrive.release.cluster.shared::cluster.b64 _, [ra];\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(cta) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t *bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAITC_%=:\n\t"
        "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONEC_%=;\n\t"
        "bra WAITC_%=;\n\t"
        "DONEC_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void umma_tf32_2sm(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n\t"
        "}" ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit_2sm(uint64_t *bar) {          // arrives at this offset in both CTAs of the pair
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(smem_u32(bar)), "h"((uint16_t)3) : "memory");
}
// 16 TMEM lanes x 8 columns per repetition; registers [4g .. 4g+3] of a lane = (row lane/4, cols 8g + 2 (lane%4) + {0,1}),
// (row lane/4 + 8, same cols)
__device__ __forceinline__ void tmem_ld_16x256b_x4(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.16x256b.x4.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr));
}
__device__ __forceinline__ void tmem_ld_16x256b_x2(uint32_t taddr, uint32_t (&v)[16]) {      // 16 columns into v[0..7]
    asm volatile("tcgen05.ld.sync.aligned.16x256b.x2.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "r"(taddr));
}

#ifdef TQC_DEVELOP
#define TQC_TRACE(a, rank, agent, it, slot) \
    do { if ((a).trace && blockIdx.x < 2 && (it) < 128) (a).trace[(((rank) * 3 + (agent)) * 128 + (it)) * 4 + (slot)] = clock64(); } while (0)
#else
#define TQC_TRACE(a, rank, agent, it, slot) do { } while (0)
#endif

__device__ __forceinline__ uint32_t tf32_nearest(uint32_t bits) { return (bits + 0x1000u) & 0xFFFFE000u; }

// NV 16-byte vectors per thread (stride TC2_SPLIT threads) of a raw tile at `addr`, lo tile `lo_ofs` bytes further.  rewrite_hi:
// hi = nearest TF32, written back in place (A); else hi = the word as the MMA reads it, truncated (B).  lo = x - hi rounded to TF32.
template <int NV, int TC2_SPLIT>
__device__ __forceinline__ void split_tile_pair(uint32_t addr, uint32_t lo_ofs, const bool rewrite_hi) {
    uint4 x[NV];
#pragma unroll
    for (int v = 0; v < NV; ++v)
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(x[v].x), "=r"(x[v].y), "=r"(x[v].z), "=r"(x[v].w)
                     : "r"(addr + (uint32_t)v * (TC2_SPLIT * 16u)));
    // the residual of a nearest-TF32 hi is signed and zero-mean, so the MMA's truncation of it is unbiased as it is; the
    // residual of a truncated hi is one-signed and is rounded to TF32 here
    auto lo_of = [&](uint32_t w, uint32_t h) {
        const uint32_t l = __float_as_uint(__uint_as_float(w) - __uint_as_float(h));
        return rewrite_hi ? l : tf32_nearest(l);
    };
#pragma unroll
    for (int v = 0; v < NV; ++v) {
        const uint32_t p = addr + (uint32_t)v * (TC2_SPLIT * 16u);
        const uint32_t rnd = rewrite_hi ? 0x1000u : 0u;
        const uint4 h = make_uint4((x[v].x + rnd) & 0xFFFFE000u, (x[v].y + rnd) & 0xFFFFE000u, (x[v].z + rnd) & 0xFFFFE000u, (x[v].w + rnd) & 0xFFFFE000u);
        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(p + lo_ofs), "r"(lo_of(x[v].x, h.x)), "r"(lo_of(x[v].y, h.y)),
                     "r"(lo_of(x[v].z, h.z)), "r"(lo_of(x[v].w, h.w)) : "memory");
        if (rewrite_hi) asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(p), "r"(h.x), "r"(h.y), "r"(h.z), "r"(h.w) : "memory");
    }
}

template <int BN>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(tc2_threads(BN), 1)
step_tc2_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, const TcArgs a) {
    constexpr int TC2_SPLIT = tc2_split_threads(BN), TC2_THREADS = tc2_threads(BN), TC2_FIRST_DRAIN = TC2_FIRST_SPLIT + TC2_SPLIT / 32;
    // the nearest-TF32 hi (rewritten in shared memory) goes to the SMALLER tile: one zero-mean residual is enough to make the
    // dropped lo*lo term unbiased, and the rewrite costs shared-memory bandwidth, the binding resource of the narrow tiles
    constexpr bool ROUND_A = BN >= 256;
    constexpr int BH = BN / 2;                       // B rows staged by one CTA
    constexpr int WC = BN / 4;                       // accumulator columns of one worker warp (4 column groups x 4 lane quadrants)
    constexpr int MAXS = 6;
    extern __shared__ unsigned char tc_smem_raw[];
    __shared__ __align__(8) uint64_t full_bar[MAXS], ready_bar[MAXS], empty_bar[MAXS], d_full_bar[2], d_empty_bar[2];
    __shared__ uint32_t tmem_base_slot;
    __shared__ uint32_t oa_mt[64], ob_nt[256], ob_c8[BN / 8];          // C-offset tables: pair m-tile, n-tile, 8-column group

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int S = a.stages;
    constexpr uint32_t bytesA = 128 * TC_BK * 4, bytesB = (uint32_t)BH * TC_BK * 4;
    constexpr uint32_t stage_bytes = 2 * bytesA + 2 * bytesB;
    unsigned char *tiles = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(tc_smem_raw) + 1023) & ~(uintptr_t)1023);
    auto A_raw = [&](int s) { return tiles + (size_t)s * stage_bytes; };
    auto A_lo = [&](int s) { return tiles + (size_t)s * stage_bytes + bytesA; };
    auto B_raw = [&](int s) { return tiles + (size_t)s * stage_bytes + 2 * bytesA; };
    auto B_lo = [&](int s) { return tiles + (size_t)s * stage_bytes + 2 * bytesA + bytesB; };

    // K = 16 (lgK = 4) runs as ONE k-block: the TMA box is 32 floats wide, the 16 beyond the tensor's K extent arrive as zeros
    const int n_kb = a.lgK >= 5 ? 1 << (a.lgK - 5) : 1;
    const int lg_tm = a.lgM - 8;
    const long long tiles_m = 1ll << lg_tm, tiles_n = (1ll << a.lgN) / BN;
    const long long total = tiles_m * tiles_n * a.R;
    const long long n_clusters = gridDim.x >> 1, cluster_id = blockIdx.x >> 1;
    const long long my_tiles = cluster_id < total ? (total - cluster_id + n_clusters - 1) / n_clusters : 0;
    const long long total_kb = my_tiles * n_kb;

    for (int x = threadIdx.x; x < 256; x += TC2_THREADS) {
        if (x < 64) oa_mt[x] = x < tiles_m ? (uint32_t)bitmap_apply(a.outA, (unsigned long long)x * TC2_BM) : 0u;
        ob_nt[x] = x < tiles_n ? (uint32_t)bitmap_apply(a.outB, (unsigned long long)x * BN) : 0u;
        if (x < BN / 8) ob_c8[x] = (uint32_t)bitmap_apply(a.outB, (unsigned long long)x * 8);
    }
    if (threadIdx.x == 0) {
        // ready / d_empty collect ONE arrival per CTA: the 16 worker warps of a CTA meet at a named barrier first (32 remote
        // arrivals on one mbarrier cost about 40 cycles each, measured: 1.2 us per k-block of pure hand-shake)
        for (int s = 0; s < S; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&ready_bar[s], 2); mbar_init(&empty_bar[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&d_full_bar[s], 1); mbar_init(&d_empty_bar[s], n_kb <= 2 ? 8 : 2); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0 && lane == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&mapB) : "memory");
    }
    if (warp == 1) {                                         // the same warp of both CTAs allocates the pair's columns
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_slot)), "r"((uint32_t)(2 * BN)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();                                      // barriers of both CTAs are initialised before any remote arrive
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem_base = tmem_base_slot;

    if (warp == 0) {
        if (lane == 0) {                                     // ===== TMA producer (each CTA loads its own rows) =====
            long long it = 0;
            for (long long t = cluster_id; t < total; t += n_clusters) {
                const long long nt = t % tiles_n, mt = (t / tiles_n) & (tiles_m - 1), r = (t / tiles_n) >> lg_tm;
                const int rowA = a.keysA ? (int)a.keysA[r] : (int)r;
                const int rowB = a.keysB ? (int)a.keysB[r] : (int)r;
                for (int kb = 0; kb < n_kb; ++kb, ++it) {
                    const int s = (int)(it % S);
                    const uint32_t ph = (uint32_t)((it / S) & 1);
                    mbar_wait(&empty_bar[s], ph ^ 1u);
                    TQC_TRACE(a, rank, 0, it, 0);
                    if (TQC_DBG(a, 64)) { mbar_arrive(&full_bar[s]); continue; }
                    mbar_expect_tx(&full_bar[s], bytesA + bytesB);
                    tma_load_3d(&mapA, &full_bar[s], A_raw(s), kb * TC_BK, (int)(mt * TC2_BM + rank * 128), rowA);
                    tma_load_3d(&mapB, &full_bar[s], B_raw(s), kb * TC_BK, (int)(nt * BN + rank * BH), rowB);
                }
            }
        }
    } else if (warp == 1) {
        if (rank == 0) {                                     // ===== MMA issuer (leader CTA) =====
            // kind::tf32, fp32 accumulate, K-major A and B, N = BN, M = 256 over the pair
            constexpr uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(BN >> 3) << 17) | ((uint32_t)(TC2_BM >> 4) << 24);
            for (long long it = 0; it < total_kb; ++it) {
                const int s = (int)(it % S);
                const uint32_t ph = (uint32_t)((it / S) & 1);
                const uint32_t db = (uint32_t)(it & 1), dph = (uint32_t)((it >> 1) & 1);
                if (!TQC_DBG(a, 256)) mbar_wait_cluster(&d_empty_bar[db], dph ^ 1u);
                if (lane == 0) TQC_TRACE(a, rank, 1, it, 0);
                mbar_wait_cluster(&ready_bar[s], ph);
                if (lane == 0) TQC_TRACE(a, rank, 1, it, 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t d_tmem = tmem_base + db * (uint32_t)BN;
                const uint64_t dah = umma_desc_sw128(smem_u32(A_raw(s))), dal = umma_desc_sw128(smem_u32(A_lo(s)));
                const uint64_t dbh = umma_desc_sw128(smem_u32(B_raw(s))), dbl = umma_desc_sw128(smem_u32(B_lo(s)));
                if (lane == 0) {
                    if (!TQC_DBG(a, 32)) {
                        // the small terms first: while the accumulator holds only lo products (2^-11 of the final value) its
                        // round-toward-zero steps are 2^-11 smaller too; only the four hi*hi accumulations see a full-size sum
#pragma unroll
                        for (int k = 0; k < TC_BK / 8; ++k) {
                            umma_tf32_2sm(d_tmem, dal + (uint64_t)(2 * k), dbh + (uint64_t)(2 * k), idesc, k ? 1u : 0u);
                            umma_tf32_2sm(d_tmem, dah + (uint64_t)(2 * k), dbl + (uint64_t)(2 * k), idesc, 1u);
                        }
#pragma unroll
                        for (int k = 0; k < TC_BK / 8; ++k) umma_tf32_2sm(d_tmem, dah + (uint64_t)(2 * k), dbh + (uint64_t)(2 * k), idesc, 1u);
                    }
                    if (TQC_DBG(a, 4096)) { mbar_arrive_cluster(&empty_bar[s], 0); mbar_arrive_cluster(&empty_bar[s], 1); }
                    else
                    umma_commit_2sm(&empty_bar[s]);              // frees the stage in both CTAs when these MMAs retire
                    if (!TQC_DBG(a, 128)) umma_commit_2sm(&d_full_bar[db]);
                    TQC_TRACE(a, rank, 1, it, 2);
                }
                __syncwarp();
            }
        }
    } else if (warp >= TC2_FIRST_SPLIT && warp < TC2_FIRST_DRAIN) {
        // ===== splitters =====
        const int st = threadIdx.x - TC2_FIRST_SPLIT * 32;
        for (long long it = 0; it < total_kb; ++it) {
            const int s = (int)(it % S);
            const uint32_t ph = (uint32_t)((it / S) & 1);
            mbar_wait(&full_bar[s], ph);
            if (st == 0) TQC_TRACE(a, rank, 2, it, 0);
            if (!TQC_DBG(a, 4)) {
                const uint32_t sa = smem_u32(A_raw(s)) + (uint32_t)st * 16u;
                constexpr int NA = (int)(bytesA >> 4) / TC2_SPLIT, NB = (int)(bytesB >> 4) / TC2_SPLIT;   // vectors per thread
                constexpr int CHA = NA < 16 ? NA : 16, CHB = NB < 16 ? NB : 16;     // all loads of a batch are in flight before the first use
                static_assert(NA % CHA == 0 && NB % CHB == 0, "tile must divide over the splitter threads");
#pragma unroll
#pragma unroll
                for (int c = 0; c < NA / CHA; ++c) split_tile_pair<CHA, TC2_SPLIT>(sa + (uint32_t)c * CHA * TC2_SPLIT * 16u, bytesA, ROUND_A);
#pragma unroll
                for (int c = 0; c < NB / CHB; ++c) split_tile_pair<CHB, TC2_SPLIT>(sa + 2u * bytesA + (uint32_t)c * CHB * TC2_SPLIT * 16u, bytesB, !ROUND_A);
            }
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");     // generic-proxy writes -> visible to the MMAs' async proxy
            asm volatile("bar.sync 1, %0;" ::"n"(TC2_SPLIT) : "memory");
            if (st == 0) { mbar_arrive_cluster(&ready_bar[s], 0); TQC_TRACE(a, rank, 2, it, 1); }
        }
    } else if (warp >= TC2_FIRST_DRAIN) {
        // ===== accumulate (round-to-nearest, registers) + store: 16 warps = 4 column groups x 4 TMEM lane quadrants =====
        const int wi = warp - TC2_FIRST_DRAIN, w4 = warp & 3, grp = wi >> 2;
        const int wt = wi * 32 + lane;
        const uint32_t lane_base = ((uint32_t)(32 * w4) << 16) + (uint32_t)(WC * grp);
        // this lane's rows of the CTA's 128 (lane/4 + 8 h, h = 0..3, inside the warp's lane quadrant) and its column pair
        uint32_t oa_row[4];
#pragma unroll
        for (int h = 0; h < 4; ++h) oa_row[h] = (uint32_t)bitmap_apply(a.outA, (unsigned long long)(rank * 128 + 32 * w4 + (lane >> 2) + 8 * h));
        const uint32_t ob_q = (uint32_t)bitmap_apply(a.outB, (unsigned long long)(2 * (lane & 3)));
        const uint32_t ob_1 = (uint32_t)bitmap_apply(a.outB, 1ull);
        const uint32_t ob_q4 = (uint32_t)bitmap_apply(a.outB, (unsigned long long)(2 * (lane & 2)));      // column 0 or 4 of a group
        long long it = 0;
        for (long long t = cluster_id; t < total; t += n_clusters) {
            const long long nt = t % tiles_n, mt = (t / tiles_n) & (tiles_m - 1), r = (t / tiles_n) >> lg_tm;
            float acc[WC];
#pragma unroll
            for (int q = 0; q < WC; ++q) acc[q] = 0.f;
            for (int kb = 0; kb < n_kb; ++kb, ++it) {
                const uint32_t db = (uint32_t)(it & 1), dph = (uint32_t)((it >> 1) & 1);
                mbar_wait(&d_full_bar[db], dph);
                if (wt == 0) TQC_TRACE(a, rank, 2, it, 2);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t taddr = tmem_base + lane_base + db * (uint32_t)BN;
                if (!TQC_DBG(a, 8)) {
                    // acc index: [half h2 (rows +16)][8-column group g][4 registers of the 16x256b pattern]
#pragma unroll
                    for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                        for (int c0 = 0; c0 < WC; c0 += 32) {
                            uint32_t v[16];
                            if (WC - c0 >= 32) tmem_ld_16x256b_x4(taddr + ((uint32_t)(16 * h2) << 16) + (uint32_t)c0, v);
                            else tmem_ld_16x256b_x2(taddr + ((uint32_t)(16 * h2) << 16) + (uint32_t)c0, v);
                            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                            for (int q = 0; q < 16; ++q)
                                if (c0 / 2 + q < WC / 2) acc[h2 * (WC / 2) + c0 / 2 + q] += __uint_as_float(v[q]);
                        }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                if (n_kb <= 2) {
                    // tiles of one or two k-blocks: one arrival per column group (4 warps, one per TMEM lane quadrant) and CTA,
                    // so that the groups may drift apart and one group's stores overlap another's drain (K = 64: -4 %,
                    // K = 16: -10 %, measured); longer tiles keep the single arrival per CTA (the extra remote arrivals cost 1-2 %)
                    asm volatile("bar.sync %0, 128;" ::"r"(2 + grp) : "memory");
                    if ((wt & 127) == 0) mbar_arrive_cluster(&d_empty_bar[db], 0);
                } else {
                    asm volatile("bar.sync 2, %0;" ::"n"(TC2_DRAIN) : "memory");
                    if (wt == 0) mbar_arrive_cluster(&d_empty_bar[db], 0);
                }
                if (wt == 0) TQC_TRACE(a, rank, 2, it, 3);
            }
            if (TQC_DBG(a, 2)) continue;
            float *ctile = a.C + r * a.c_row_stride + (oa_mt[mt] | ob_nt[nt]);
            if (a.vec4 == 2) {
                // columns c .. c+3 (c a multiple of 4) are neighbours in C: neighbouring lanes of a quad swap halves of two
                // 8-column groups, so that an even lane holds 4 consecutive columns of group g, the odd lane next to it 4 of
                // group g + 1, and a lane stores 16 bytes: a quad writes 64 contiguous bytes of a row where the layout allows
                // (the store path alone, all SMs, profiles/peaks_r02.md: 5.5 TB/s for both at a row pitch of 16 KB, 5.5 against
                // 5.1 for 8-byte stores at 64 KB, 3.1 against 1.5 at 1 MB; in the kernel: -2 to -3 % on K <= 256 steps)
                const bool odd = (lane & 1) != 0;
#pragma unroll
                for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                    for (int g = 0; g < WC / 8; g += 2) {
                        const float *e = &acc[h2 * (WC / 2) + 4 * g], *o = e + 4;
                        const float r0 = __shfl_xor_sync(0xffffffffu, odd ? e[0] : o[0], 1), r1 = __shfl_xor_sync(0xffffffffu, odd ? e[1] : o[1], 1);
                        const float r2 = __shfl_xor_sync(0xffffffffu, odd ? e[2] : o[2], 1), r3 = __shfl_xor_sync(0xffffffffu, odd ? e[3] : o[3], 1);
                        const uint32_t oc = ob_c8[grp * (WC / 8) + g + (odd ? 1 : 0)] | ob_q4;
                        *reinterpret_cast<float4 *>(ctile + (oa_row[2 * h2] | oc)) = odd ? make_float4(r0, r1, o[0], o[1]) : make_float4(e[0], e[1], r0, r1);
                        *reinterpret_cast<float4 *>(ctile + (oa_row[2 * h2 + 1] | oc)) = odd ? make_float4(r2, r3, o[2], o[3]) : make_float4(e[2], e[3], r2, r3);
                    }
                continue;
            }
#pragma unroll
            for (int h2 = 0; h2 < 2; ++h2)
#pragma unroll
                for (int g = 0; g < WC / 8; ++g) {
                    const uint32_t oc = ob_c8[grp * (WC / 8) + g] | ob_q;
                    const float *v4 = &acc[h2 * (WC / 2) + 4 * g];            // (row, c), (row, c+1), (row+8, c), (row+8, c+1)
                    float *p0 = ctile + (oa_row[2 * h2] | oc), *p1 = ctile + (oa_row[2 * h2 + 1] | oc);
                    if (a.vec4) {                                             // columns c, c+1 are neighbours in C
                        *reinterpret_cast<float2 *>(p0) = make_float2(v4[0], v4[1]);
                        *reinterpret_cast<float2 *>(p1) = make_float2(v4[2], v4[3]);
                    } else {
                        p0[0] = v4[0]; p0[ob_1] = v4[1];
                        p1[0] = v4[2]; p1[ob_1] = v4[3];
                    }
                }
        }
    }

    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    cluster_sync_all();                                      // no CTA leaves while its peer may still signal it
    if (warp == 1) {
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"((uint32_t)(2 * BN)) : "memory");
    }
}

}  // namespace tqc
