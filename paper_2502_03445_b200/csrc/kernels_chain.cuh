// Fused small-bond chain (sm_100a): when every per-state step of a plan is small, the whole per-state tail of the
// contraction tree — gathers (a3), pairwise contractions (a4) and the final reduction (a5) —
// runs in ONE kernel, one warp per state, with every intermediate kept in that warp's shared memory instead of
// round-tripping through HBM.  Bond sums that have fewer than 32 outputs are split over lanes and finished with warp
// shuffles.  The step table is plan data (built once on the host, read from global memory).
#pragma once
#if !defined(__CUDACC_RTC__)
#include <cuda_runtime.h>
#include <stdint.h>
#endif

#include "device_args.h"

namespace tqc {

constexpr int CHAIN_MAX_STEPS = 24;
constexpr int CHAIN_WARPS = 8;                 // warps (states in flight) per block

constexpr int CHAIN_MAX_GATHER = 16;
constexpr int CHAIN_MAX_F4 = 6;                // float4 vectors per lane of one state's staged operands (768 floats)

struct ChainOperand {
    const float *base;       // LEAF: its device tensor (rows of 2^{lgRows+lgK} floats)
    long long table_ofs;     // TABLE: float offset inside the workspace's table region (-1 otherwise)
    int gathered;            // 1: LEAF or TABLE row selected by the state's key; 0: intermediate in shared memory
    int key_slot;            // gathered: row = keys[key_slot * cap + r]
    int smem_ofs;            // float offset in the warp's scratch (staged gather or intermediate)
    int staged;              // gathered operand copied to shared memory at the start of the state
    int pitch;               // floats between consecutive rows where the inner loop reads it (K, or K + 4 in shared memory)
};

struct ChainStep {
    ChainOperand A, B;
    int lgM, lgN, lgK;
    int c_smem_ofs;          // result: float offset in the warp's scratch, or -1: the root, written to out[r]
    int c_lgK;               // log2 of the row length the consumer reads the result with (rows are padded by 4 floats)
    int tab_ofs;             // offset of this step's index tables in the block's u16 table area: [M entries][N entries]
    BitMap outA, outB;       // i -> bits of the result's linear index, j -> bits (disjoint)
};

struct ChainGather {         // one staged operand: all of them are fetched together when a warp starts a state
    const float *base;
    long long table_ofs;
    int key_slot, lg_floats, lgK, smem_ofs, f4_begin;
};

struct ChainArgs {
    const ChainStep *steps;  // DEVICE [n_steps]
    int n_steps;
    int n_slots;             // key slots of the plan (<= 32 for the chain kernel)
    int n_gather, total_f4;
    ChainGather g[CHAIN_MAX_GATHER];
    const float *tables;     // states-mode table region of the workspace
    const uint32_t *keys;    // [n_slots][cap]
    long long cap;
    float *out;
    int R;
    int scratch_floats;      // per warp: [stage buffer 0][stage buffer 1][intermediates]
    int stage_floats;        // one stage buffer (all staged operands of one state)
    int tab_entries;         // u16 index-table entries per block
};

// index of element x of a padded intermediate: rows of 2^lgK floats, 4 floats of padding per row (bank spread for float4 reads)
__device__ __forceinline__ int chain_pad(int x, int lgK) { return lgK >= 2 ? x + ((x >> lgK) << 2) : x; }

// KS floats of the bond per lane and output: fully unrolled float4 loads for the common small bonds
template <int KS>
__device__ __forceinline__ float dot_fixed(const float *pa, const float *pb) {
    if (KS < 4) {
        float s = 0.f;
#pragma unroll
        for (int k = 0; k < KS; ++k) s = fmaf(pa[k], pb[k], s);
        return s;
    }
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
#pragma unroll
    for (int k = 0; k < KS; k += 4) {
        const float4 x = *reinterpret_cast<const float4 *>(pa + k), y = *reinterpret_cast<const float4 *>(pb + k);
        s0 = fmaf(x.x, y.x, s0); s1 = fmaf(x.y, y.y, s1); s2 = fmaf(x.z, y.z, s2); s3 = fmaf(x.w, y.w, s3);
    }
    return (s0 + s1) + (s2 + s3);
}

struct ChainStepCtx {           // per-step values every pass of the output loop needs
    const float *pa, *pb;
    const uint16_t *ta, *tb;
    float *scr, *out_r;
    int pitchA, pitchB, lgN, lgO, lgG, c_smem_ofs, c_lgK, lane;
};

// all outputs of one step for one state; KS = bond floats per lane (K / G), a multiple of 64 loops over 64-float pieces
template <int KS>
__device__ __forceinline__ void chain_outputs(const ChainStepCtx &c, int kspan) {
    const int G = 1 << c.lgG, g = c.lane & (G - 1), per_pass = 32 >> c.lgG, n_out = 1 << c.lgO, nmask = (1 << c.lgN) - 1;
    for (int o0 = 0; o0 < n_out; o0 += per_pass) {
        const int o = o0 + (c.lane >> c.lgG);
        const bool live = o < n_out;
        const int i = o >> c.lgN, j = o & nmask;
        float v = 0.f;
        if (live) {
            const float *qa = c.pa + i * c.pitchA + g * kspan, *qb = c.pb + j * c.pitchB + g * kspan;
            if (KS <= 64) v = dot_fixed<KS>(qa, qb);
            else for (int k = 0; k < kspan; k += 64) v += dot_fixed<64>(qa + k, qb + k);
        }
        for (int d = G >> 1; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
        if (live && g == 0) {
            if (c.c_smem_ofs < 0) *c.out_r = v;
            else c.scr[c.c_smem_ofs + chain_pad((int)(c.ta[i] | c.tb[j]), c.c_lgK)] = v;
        }
    }
}

// Plan-specialised step (used by the run-time generated Spec): M = 2^LGM, N = 2^LGN, K = 2^LGK and both row pitches are
// compile-time constants, so every loop unrolls and the index arithmetic folds away.  With >= 32 outputs a lane owns the
// outputs o = lane + 32 p; they form an NI x NJ grid (NJ distinct j, NI distinct i) whose operand rows are loaded once per
// 16-float slab of the bond and reused from registers.  With fewer outputs the bond is split over G lanes per output and
// finished with warp shuffles.  emit(i, j, value) stores one result.
// x = hi + lo with hi the nearest TF32 and lo the exact remainder (the tensor core reads its top 19 bits): the operands of
// a 3xTF32 product
__device__ __forceinline__ void tf32_split(float x, uint32_t &hi, uint32_t &lo) {
    hi = (__float_as_uint(x) + 0x1000u) & 0xFFFFE000u;          // round-to-nearest TF32 of a finite x
    lo = __float_as_uint(x - __uint_as_float(hi));              // exact remainder
#if defined(TQC_MMA_MASK_LO)
    lo &= 0xFFFFE000u;                                          // what the tensor core does with the low 13 bits anyway
#endif
}
__device__ __forceinline__ void mma_tf32_16x8x8(float (&d)[4], const uint32_t (&a)[4], const uint32_t (&b)[2]) {
    asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}

// Warp-level tensor-core step for the larger outputs of a chain (M >= 16, N >= 8, K >= 8; at most 1024 outputs): the warp's
// one state is an M x N x K product small enough for mma.sync fragments, far too small for a tcgen05 tile.  3xTF32
// (lo*hi + hi*lo + hi*hi, fp32 accumulate); each lane loads 4 A and 2 B scalars per 16x8x8 block from the K-major rows
// (conflict-free with the 4-float row pad) and splits them once per k-step.
// SLICE_SUM: see the comment at the MMAs.  The table steps (kernels_cross.cuh) feed one another - cfg5 runs 24 in a row -
// and take the slice sums; a chain's one product per state keeps the running accumulator (cfg4: mean error -5e-8 of max p,
// and the extra adds cost 1.5 % of the chain kernel).
// the accumulators only: acc[mi][nj] = {(row 16 mi + g, col 8 nj + 2 t), (same row, col + 1), (row + 8, col), (row + 8, col + 1)}
template <int LGM, int LGN, int LGK, int PA, int PB, bool SLICE_SUM = false>
__device__ __forceinline__ void chain_mma_acc(const float *pa, const float *pb, int lane, float (&acc)[(1 << LGM) / 16][(1 << LGN) / 8][4]) {
    constexpr int MT = (1 << LGM) / 16, NT = (1 << LGN) / 8, K = 1 << LGK;
    const int g = lane >> 2, t = lane & 3;
#pragma unroll
    for (int mi = 0; mi < MT; ++mi)
#pragma unroll
        for (int nj = 0; nj < NT; ++nj)
#pragma unroll
            for (int e = 0; e < 4; ++e) acc[mi][nj][e] = 0.f;
#pragma unroll
    for (int k0 = 0; k0 < K; k0 += 8) {
        uint32_t ah[MT][4], al[MT][4], bh[NT][2], bl[NT][2];
#pragma unroll
        for (int mi = 0; mi < MT; ++mi) {
            const float *p = pa + (mi * 16 + g) * PA + k0 + t;
            tf32_split(p[0], ah[mi][0], al[mi][0]);
            tf32_split(p[8 * PA], ah[mi][1], al[mi][1]);
            tf32_split(p[4], ah[mi][2], al[mi][2]);
            tf32_split(p[8 * PA + 4], ah[mi][3], al[mi][3]);
        }
#pragma unroll
        for (int nj = 0; nj < NT; ++nj) {
            const float *q = pb + (nj * 8 + g) * PB + k0 + t;
            tf32_split(q[0], bh[nj][0], bl[nj][0]);
            tf32_split(q[4], bh[nj][1], bl[nj][1]);
        }
#pragma unroll
        for (int mi = 0; mi < MT; ++mi)
#pragma unroll
            for (int nj = 0; nj < NT; ++nj) {
                // the tensor pipe truncates its accumulator (measured: DESIGN.md 5.3), so a running sum kept there drifts
                // by about -0.5 ulp per MMA.  With SLICE_SUM each bond slice is summed from zero (small terms first: one
                // truncation at the slice's own magnitude) and joins the running sum in registers, rounded to nearest.
                if constexpr (SLICE_SUM) {
                    float d[4] = {0.f, 0.f, 0.f, 0.f};
                    mma_tf32_16x8x8(d, al[mi], bh[nj]);
                    mma_tf32_16x8x8(d, ah[mi], bl[nj]);
                    mma_tf32_16x8x8(d, ah[mi], bh[nj]);
#pragma unroll
                    for (int e = 0; e < 4; ++e) acc[mi][nj][e] += d[e];
                } else {
                    mma_tf32_16x8x8(acc[mi][nj], al[mi], bh[nj]);       // small terms first
                    mma_tf32_16x8x8(acc[mi][nj], ah[mi], bl[nj]);
                    mma_tf32_16x8x8(acc[mi][nj], ah[mi], bh[nj]);
                }
            }
    }
}

template <int LGM, int LGN, int LGK, int PA, int PB, bool SLICE_SUM = false, class Emit>
__device__ __forceinline__ void chain_step_mma(const float *pa, const float *pb, int lane, Emit emit) {
    constexpr int MT = (1 << LGM) / 16, NT = (1 << LGN) / 8;
    const int g = lane >> 2, t = lane & 3;
    float acc[MT][NT][4];
    chain_mma_acc<LGM, LGN, LGK, PA, PB, SLICE_SUM>(pa, pb, lane, acc);
#pragma unroll
    for (int mi = 0; mi < MT; ++mi)
#pragma unroll
        for (int nj = 0; nj < NT; ++nj) {
            emit(mi * 16 + g, nj * 8 + 2 * t, acc[mi][nj][0]);
            emit(mi * 16 + g, nj * 8 + 2 * t + 1, acc[mi][nj][1]);
            emit(mi * 16 + g + 8, nj * 8 + 2 * t, acc[mi][nj][2]);
            emit(mi * 16 + g + 8, nj * 8 + 2 * t + 1, acc[mi][nj][3]);
        }
}

template <int LGM, int LGN, int LGK, int PA, int PB, bool ROWSPLIT = false, class Emit>
__device__ __forceinline__ void chain_step_spec(const float *pa, const float *pb, int lane, Emit emit) {
    constexpr int N = 1 << LGN, K = 1 << LGK, LGO = LGM + LGN, O = 1 << LGO;
#if !defined(TQC_CHAIN_NO_MMA)
    if constexpr (!ROWSPLIT && LGK >= 3 && LGO <= 10 && LGM >= 4 && LGN >= 3) {
        chain_step_mma<LGM, LGN, LGK, PA, PB>(pa, pb, lane, emit);
        return;
    } else if constexpr (!ROWSPLIT && LGK >= 3 && LGO <= 10 && LGN >= 4 && LGM >= 3) {
        chain_step_mma<LGN, LGM, LGK, PB, PA>(pb, pa, lane, [&](int j, int i, float v) { emit(i, j, v); });
        return;
    }
#endif
    if constexpr (ROWSPLIT) {
        // M == 1 and B is read straight from global memory (each element is used once per state): out[j] = sum_k a[k] B[j][k].
        // The lanes split the bond so that every load of B is a contiguous 16 B x G segment of one row (coalesced), the
        // partial sums of a row meet by warp shuffles.
        static_assert(LGM == 0 && LGK >= 4, "row-split step");
        constexpr int G = K / 4 < 32 ? K / 4 : 32;          // lanes per row
        constexpr int RP = 32 / G;                           // rows per pass
        constexpr int NQ = K / (4 * G);                      // float4 per lane per row
        const int g = lane % G, rr = lane / G;
        float4 a4[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) a4[q] = *reinterpret_cast<const float4 *>(pa + 4 * g + 4 * G * q);
        // U passes (U * RP rows) per round: all their loads are issued before the first use (the step is bound by the
        // latency of these L2 reads, not by their bandwidth), and the U partial sums of a lane meet their G - 1 partners by
        // recursive halving - each level a lane keeps half of its values and sends the other half - so U rows cost about
        // U shuffles instead of U log2 G.  Lane g ends with the row whose pass number is the top log2 U bits of g.
        constexpr int UMAX = NQ >= 8 ? 1 : 8 / NQ;
        constexpr int U = G < UMAX ? G : UMAX;
        constexpr int LGG = G == 32 ? 5 : G == 16 ? 4 : G == 8 ? 3 : 2, LGU = U == 8 ? 3 : U == 4 ? 2 : U == 2 ? 1 : 0;
        static_assert((1 << LGG) == G && (1 << LGU) == U, "row-split lane groups");
#pragma unroll 1
        for (int jb = 0; jb < N; jb += U * RP) {
            float4 b[U][NQ];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const int j = jb + u * RP + rr;
#pragma unroll
                for (int q = 0; q < NQ; ++q)
                    b[u][q] = j < N ? __ldg(reinterpret_cast<const float4 *>(pb + (size_t)j * PB + 4 * g + 4 * G * q))
                                    : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            float v[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                float s0 = 0.f, s1 = 0.f;
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    s0 = fmaf(a4[q].x, b[u][q].x, s0); s1 = fmaf(a4[q].y, b[u][q].y, s1);
                    s0 = fmaf(a4[q].z, b[u][q].z, s0); s1 = fmaf(a4[q].w, b[u][q].w, s1);
                }
                v[u] = s0 + s1;
            }
            int cnt = U;
#pragma unroll
            for (int d = G >> 1; d > 0; d >>= 1) {
                if (cnt > 1) {
                    const bool up = (g & d) != 0;
#pragma unroll
                    for (int i = 0; i < cnt / 2; ++i) {
                        const float send = up ? v[i] : v[i + cnt / 2];
                        const float keep = up ? v[i + cnt / 2] : v[i];
                        v[i] = keep + __shfl_xor_sync(0xffffffffu, send, d);
                    }
                    cnt /= 2;
                } else {
                    v[0] += __shfl_xor_sync(0xffffffffu, v[0], d);
                }
            }
            const int j = jb + (g >> (LGG - LGU)) * RP + rr;
            if (j < N && (g & ((1 << (LGG - LGU)) - 1)) == 0) emit(0, j, v[0]);
        }
    } else if constexpr (O >= 32 && LGK >= 2) {
        // a lane owns an NI x NJ block of outputs: rows i0 + x * SI, columns j0 + y * SJ, with the 32 lanes laid out LI x LJ
        // over the M x N outputs.  Shared-memory traffic per lane is (NI + NJ) rows per bond slab, so the block is kept as
        // square as the shape allows (16 x 16 outputs: 2 x 4 instead of 8 x 1, a third fewer loads).
        constexpr int M = 1 << LGM, PER = O / 32;
        constexpr int LGPER = LGO - 5;
        constexpr int LGNJ0 = (LGPER + 1) / 2;                                     // aim for NJ >= NI
        constexpr int LGNJ = LGNJ0 > LGN ? LGN : (LGPER - LGNJ0 > LGM ? LGPER - LGM : LGNJ0);
        constexpr int NJ = 1 << LGNJ, NI = PER / NJ;
        constexpr int LJ = N / NJ, LI = M / NI;                                    // lane grid, LI * LJ == 32
        static_assert(LI * LJ == 32 && NI * NJ == PER, "lane tiling");
        constexpr int KC = K < 16 ? K : 16;
        const int j0 = lane % LJ, i0 = lane / LJ;
        float acc[NI][NJ];
#pragma unroll
        for (int x = 0; x < NI; ++x)
#pragma unroll
            for (int y = 0; y < NJ; ++y) acc[x][y] = 0.f;
#pragma unroll
        for (int k0 = 0; k0 < K; k0 += KC) {
            float4 b[NJ][KC / 4];
#pragma unroll
            for (int y = 0; y < NJ; ++y)
#pragma unroll
                for (int q = 0; q < KC / 4; ++q) b[y][q] = *reinterpret_cast<const float4 *>(pb + (j0 + LJ * y) * PB + k0 + 4 * q);
#pragma unroll
            for (int x = 0; x < NI; ++x) {
#pragma unroll
                for (int q = 0; q < KC / 4; ++q) {
                    const float4 av = *reinterpret_cast<const float4 *>(pa + (i0 + LI * x) * PA + k0 + 4 * q);
#pragma unroll
                    for (int y = 0; y < NJ; ++y) {
                        acc[x][y] = fmaf(av.x, b[y][q].x, acc[x][y]); acc[x][y] = fmaf(av.y, b[y][q].y, acc[x][y]);
                        acc[x][y] = fmaf(av.z, b[y][q].z, acc[x][y]); acc[x][y] = fmaf(av.w, b[y][q].w, acc[x][y]);
                    }
                }
            }
        }
#pragma unroll
        for (int x = 0; x < NI; ++x)
#pragma unroll
            for (int y = 0; y < NJ; ++y) emit(i0 + LI * x, j0 + LJ * y, acc[x][y]);
    } else {
        constexpr int LGG0 = LGO >= 5 ? 0 : 5 - LGO;
        constexpr int LGG = (LGK - LGG0 < 2) ? (LGK >= 2 ? LGK - 2 : 0) : LGG0;
        constexpr int G = 1 << LGG, KS = K >> LGG, PASS = 32 >> LGG;
        const int g = lane & (G - 1);
#pragma unroll
        for (int o0 = 0; o0 < O; o0 += PASS) {
            const int o = o0 + (lane >> LGG);
            const bool live = o < O;
            const int i = o >> LGN, j = o & (N - 1);
            float v = 0.f;
            if (live) {
#pragma unroll
                for (int k = 0; k < KS; k += 64)
                    v += dot_fixed<(KS - 0 < 64 ? KS : 64)>(pa + i * PA + g * KS + k, pb + j * PB + g * KS + k);
            }
#pragma unroll
            for (int d = G >> 1; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (live && g == 0) emit(i, j, v);
        }
    }
}

__device__ __forceinline__ void chain_cp16(uint32_t dst_smem, const float *src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");   // .ca measured slower
}

// what a state's steps see: the warp's stage buffer of the current state, its intermediates, this state's keys (one per lane)
struct ChainStateCtx {
    const ChainArgs *a;
    const ChainStep *steps;     // shared-memory copy of the step table
    const uint16_t *tabs;       // result-index tables
    const float *stg;
    float *inter, *out_r;
    uint32_t mykey;
    int lane;
};

// Spec::run(ctx) executes every step of the plan for one state.  ChainInterp walks the step table; a plan-specialised Spec
// (generated and compiled at run time by the library, chain_jit.cpp) has the same steps as straight-line code.
template <class Spec>
__device__ __forceinline__ void chain_body(const ChainArgs &a) {
    extern __shared__ __align__(16) unsigned char chain_smem_raw[];
    // block layout: [step table][u16 index tables][per-warp scratch]
    ChainStep *steps = reinterpret_cast<ChainStep *>(chain_smem_raw);
    const size_t steps_bytes = ((size_t)a.n_steps * sizeof(ChainStep) + 15) & ~(size_t)15;
    uint16_t *tabs = reinterpret_cast<uint16_t *>(chain_smem_raw + steps_bytes);
    const size_t tabs_bytes = ((size_t)a.tab_entries * 2 + 15) & ~(size_t)15;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // gather table: for float4 number f of a state's staged operands: {source base, key slot, log2 row floats, float offset in
    // the row, destination in the warp scratch} — the same for every state
    uint4 *gtab = reinterpret_cast<uint4 *>(chain_smem_raw + steps_bytes + tabs_bytes);
    const size_t gtab_bytes = (size_t)a.total_f4 * sizeof(uint4);
    float *scr = reinterpret_cast<float *>(chain_smem_raw + steps_bytes + tabs_bytes + gtab_bytes) + (size_t)warp * a.scratch_floats;

    {   // once per block: step table and result-index tables into shared memory
        const uint32_t *src = reinterpret_cast<const uint32_t *>(a.steps);
        uint32_t *dst = reinterpret_cast<uint32_t *>(steps);
        for (int x = threadIdx.x; x < (int)(a.n_steps * sizeof(ChainStep) / 4); x += blockDim.x) dst[x] = src[x];
        __syncthreads();
        for (int t = 0; t < a.n_steps; ++t) {
            const ChainStep &s = steps[t];
            const int M = 1 << s.lgM, N = 1 << s.lgN;
            for (int x = threadIdx.x; x < M + N; x += blockDim.x)
                tabs[s.tab_ofs + x] = (uint16_t)(x < M ? bitmap_apply(s.outA, (unsigned long long)x) : bitmap_apply(s.outB, (unsigned long long)(x - M)));
        }
        for (int f = threadIdx.x; f < a.total_f4; f += blockDim.x) {
            int gi = 0;
            for (int x = 1; x < a.n_gather; ++x) if (f >= a.g[x].f4_begin) gi = x;
            const ChainGather &gg = a.g[gi];
            const int x = (f - gg.f4_begin) * 4;
            const unsigned long long src = (unsigned long long)((gg.table_ofs >= 0 ? a.tables + gg.table_ofs : gg.base) + x);
            gtab[f] = make_uint4((uint32_t)src, (uint32_t)(src >> 32), (uint32_t)gg.key_slot | ((uint32_t)gg.lg_floats << 8),
                                 (uint32_t)(gg.smem_ofs + chain_pad(x, gg.lgK)));
        }
        __syncthreads();
    }

    const long long n_warps = (long long)gridDim.x * CHAIN_WARPS;
    // software pipeline over this warp's states: keys are fetched two states ahead; the staged operands of the NEXT state
    // are copied global -> shared by cp.async into the other stage buffer while the current state computes, so neither
    // registers nor the critical path carry the gather latency
    auto load_key = [&](long long rr) -> uint32_t {
        return (rr < a.R && lane < a.n_slots) ? a.keys[(long long)lane * a.cap + rr] : 0u;
    };
    float *inter = scr + 2 * a.stage_floats;
    auto issue_gather = [&](uint32_t key_of_state, int buf) {
        const uint32_t dst_base = (uint32_t)__cvta_generic_to_shared(scr + buf * a.stage_floats);
        if constexpr (Spec::kOwnGather) {                                    // plan-specialised: straight-line copies
            Spec::gather(a, key_of_state, dst_base, lane);
            asm volatile("cp.async.commit_group;" ::: "memory");
            return;
        }
#pragma unroll
        for (int q = 0; q < CHAIN_MAX_F4; ++q) {
            if (q * 32 < a.total_f4) {                                       // uniform
                const uint4 e = gtab[min(q * 32 + lane, a.total_f4 - 1)];
                const uint32_t key = __shfl_sync(0xffffffffu, key_of_state, e.z & 31u);
                const float *src = reinterpret_cast<const float *>((unsigned long long)e.x | ((unsigned long long)e.y << 32)) +
                                   ((size_t)key << (e.z >> 8));
                if (q * 32 + lane < a.total_f4)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_base + e.w * 4u), "l"(src) : "memory");
            }
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };
    const long long r0 = (long long)blockIdx.x * CHAIN_WARPS + warp;
    uint32_t mykey = load_key(r0), key_n1 = load_key(r0 + n_warps);
    if (r0 < a.R) issue_gather(mykey, 0);
    int buf = 0;
    for (long long r = r0; r < a.R; r += n_warps, buf ^= 1) {
        const uint32_t key_n2 = load_key(r + 2 * n_warps);
        __syncwarp();                                                   // the previous state's readers are done with the other buffer
        if (r + n_warps < a.R) {
            issue_gather(key_n1, buf ^ 1);                              // in flight while this state computes
            asm volatile("cp.async.wait_group 1;" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;" ::: "memory");
        }
        __syncwarp();
        const float *stg = scr + buf * a.stage_floats;
        ChainStateCtx sc;
        sc.a = &a; sc.steps = steps; sc.tabs = tabs; sc.stg = stg; sc.inter = inter; sc.out_r = a.out + r; sc.mykey = mykey; sc.lane = lane;
        Spec::run(sc);
        mykey = key_n1; key_n1 = key_n2;
    }
}

struct ChainInterp {
    static constexpr bool kOwnGather = false;
    static __device__ __forceinline__ void gather(const ChainArgs &, uint32_t, uint32_t, int) {}
    static __device__ __forceinline__ void run(const ChainStateCtx &sc) {
        const ChainArgs &a = *sc.a;
        for (int t = 0; t < a.n_steps; ++t) {
            const ChainStep &s = sc.steps[t];
            const int K = 1 << s.lgK;
            const float *pa, *pb;
            if (!s.A.gathered) pa = sc.inter + s.A.smem_ofs;
            else if (s.A.staged) pa = sc.stg + s.A.smem_ofs;
            else pa = (s.A.table_ofs >= 0 ? a.tables + s.A.table_ofs : s.A.base) +
                      ((size_t)__shfl_sync(0xffffffffu, sc.mykey, s.A.key_slot) << (s.lgM + s.lgK));
            if (!s.B.gathered) pb = sc.inter + s.B.smem_ofs;
            else if (s.B.staged) pb = sc.stg + s.B.smem_ofs;
            else pb = (s.B.table_ofs >= 0 ? a.tables + s.B.table_ofs : s.B.base) +
                      ((size_t)__shfl_sync(0xffffffffu, sc.mykey, s.B.key_slot) << (s.lgN + s.lgK));
            // ---- outputs: G lanes share one output when there are fewer than 32 of them ----
            ChainStepCtx c;
            c.pa = pa; c.pb = pb; c.pitchA = s.A.pitch; c.pitchB = s.B.pitch;
            c.lgN = s.lgN; c.lgO = s.lgM + s.lgN;
            c.lgG = c.lgO >= 5 ? 0 : 5 - c.lgO;
            if (s.lgK - c.lgG < 2) c.lgG = s.lgK >= 2 ? s.lgK - 2 : 0;        // at least one float4 of the bond per lane
            c.ta = sc.tabs + s.tab_ofs; c.tb = c.ta + (1 << s.lgM);
            c.scr = sc.inter; c.out_r = sc.out_r; c.c_smem_ofs = s.c_smem_ofs; c.c_lgK = s.c_lgK; c.lane = sc.lane;
            const int kspan = K >> c.lgG;
            switch (kspan) {
                case 1: chain_outputs<1>(c, kspan); break;
                case 4: chain_outputs<4>(c, kspan); break;
                case 8: chain_outputs<8>(c, kspan); break;
                case 16: chain_outputs<16>(c, kspan); break;
                case 32: chain_outputs<32>(c, kspan); break;
                case 64: chain_outputs<64>(c, kspan); break;
                default: chain_outputs<128>(c, kspan); break;
            }
            __syncwarp();
        }
    }
};

#if !defined(__CUDACC_RTC__)
__global__ void __launch_bounds__(CHAIN_WARPS * 32, 3) chain_kernel(const ChainArgs a) { chain_body<ChainInterp>(a); }
#endif

}  // namespace tqc
