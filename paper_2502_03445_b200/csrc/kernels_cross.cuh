// Table steps with a short bond (K = 8 .. 64) and many rows on both sides: the cross-mode contraction of a4/a6
//     C[outA(i') | outB(j')] = sum_k A[rowA(i'), k] * B[rowB(j'), k]
// is one M' x N' x K product per step (PAPER.md lines 318-330 merged bond).  With K this
// short the fp32 FFMA kernel is bound by instruction issue, not by the result write, so the products run on the tensor
// pipe as warp-level 3xTF32 mma.sync blocks (kernels_chain.cuh: chain_step_mma, one bond slice of 8 per accumulator and the
// slices added in registers: table steps feed one another and the pipe's truncating accumulator would drift), 64 x 128
// outputs per 256-thread block.
// Where j' and j' + 1 are neighbours in C (the usual case: the result layout keeps the operand's digit order) the results
// leave straight from the fragments as 8-byte stores, four lanes per 32-byte sector; otherwise the tile goes through
// shared memory and leaves row by row.
#pragma once
#include "device_args.h"
#include "kernels_chain.cuh"

namespace tqc {

constexpr int CROSS_TI = 64, CROSS_TJ = 128, CROSS_CP = CROSS_TJ + 8;      // C tile pitch (floats)

template <int LGK>
__global__ void __launch_bounds__(256, LGK >= 5 ? 3 : 4) cross_mma_kernel(const StepArgs a) {     // K >= 32: 64 registers spill (slice sums)
    constexpr int K = 1 << LGK, P = K + 4;                                // row pitch: fragment loads hit 32 distinct banks
    extern __shared__ __align__(16) unsigned char cross_smem_raw[];
    unsigned long long *rowA = reinterpret_cast<unsigned long long *>(cross_smem_raw);   // [TI] operand row offsets (floats)
    unsigned long long *rowB = rowA + CROSS_TI;                                           // [TJ]
    unsigned long long *offA = rowB + CROSS_TJ;                                           // [TI] C offset bits of i'
    unsigned long long *offB = offA + CROSS_TI;                                           // [TJ] C offset bits of j'
    float *As = reinterpret_cast<float *>(offB + CROSS_TJ);                               // [TI][P]
    float *Bs = As + CROSS_TI * P;                                                        // [TJ][P]
    float *Cs = Bs + CROSS_TJ * P;                                                        // [TI][CROSS_CP]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long bid = blockIdx.x;
    const unsigned long long tjb = (unsigned long long)(bid & ((1ll << a.lgTilesJ) - 1));
    const unsigned long long tib = (unsigned long long)(bid >> a.lgTilesJ);

    if (tid < CROSS_TI) {
        const unsigned long long ip = tib * CROSS_TI + tid;
        rowA[tid] = (a.A.use_map ? (bitmap_apply(a.A.in_map, ip) | a.A.in_or) : ip) << LGK;
        offA[tid] = bitmap_apply(a.outA, ip);
    }
    if (tid >= 128) {
        const int j = tid - 128;
        const unsigned long long jp = tjb * CROSS_TJ + j;
        rowB[j] = (a.B.use_map ? (bitmap_apply(a.B.in_map, jp) | a.B.in_or) : jp) << LGK;
        offB[j] = bitmap_apply(a.outB, jp);
    }
    __syncthreads();
    for (int e = tid; e < CROSS_TI * (K / 4); e += 256) {
        const int row = e >> (LGK - 2), k4 = e & (K / 4 - 1);
        *reinterpret_cast<float4 *>(As + row * P + 4 * k4) = __ldg(reinterpret_cast<const float4 *>(a.A.base + rowA[row]) + k4);
    }
    for (int e = tid; e < CROSS_TJ * (K / 4); e += 256) {
        const int row = e >> (LGK - 2), k4 = e & (K / 4 - 1);
        *reinterpret_cast<float4 *>(Bs + row * P + 4 * k4) = __ldg(reinterpret_cast<const float4 *>(a.B.base + rowB[row]) + k4);
    }
    __syncthreads();
    if (a.vec_store == 2) {
        // j' and j' + 1 are neighbours in C: the two results a lane holds per fragment row leave as one 8-byte store, four
        // lanes fill a 32-byte sector, no trip through shared memory
        const int wi = warp >> 2, wj = warp & 3;
        float keep = 0.f;
        chain_step_mma<5, 5, LGK, P, P, true>(As + 32 * wi * P, Bs + 32 * wj * P, lane, [&](int i, int j, float v) {
            if ((j & 1) == 0) keep = v;
            else *reinterpret_cast<float2 *>(a.C + (offA[32 * wi + i] | offB[32 * wj + j - 1])) = make_float2(keep, v);
        });
        return;
    }
    {   // warp grid 2 x 4 over the 64 x 128 tile: 32 x 32 outputs per warp
        const int wi = warp >> 2, wj = warp & 3;
        float *cw = Cs + (32 * wi) * CROSS_CP + 32 * wj;
        chain_step_mma<5, 5, LGK, P, P, true>(As + 32 * wi * P, Bs + 32 * wj * P, lane, [&](int i, int j, float v) { cw[i * CROSS_CP + j] = v; });
    }
    __syncthreads();
    for (int e = tid; e < CROSS_TI * (CROSS_TJ / 4); e += 256) {
        const int i = e >> 5, j4 = (e & 31) * 4;
        const float4 v = *reinterpret_cast<const float4 *>(Cs + i * CROSS_CP + j4);
        const unsigned long long oa = offA[i];
        if (a.vec_store) *reinterpret_cast<float4 *>(a.C + (oa | offB[j4])) = v;
        else {
            a.C[oa | offB[j4]] = v.x; a.C[oa | offB[j4 + 1]] = v.y; a.C[oa | offB[j4 + 2]] = v.z; a.C[oa | offB[j4 + 3]] = v.w;
        }
    }
}

inline size_t cross_mma_smem(int lgK, bool staged_c) {
    const size_t P = ((size_t)1 << lgK) + 4;
    return 8 * 2 * (size_t)(CROSS_TI + CROSS_TJ) + 4 * (size_t)(CROSS_TI + CROSS_TJ) * P + (staged_c ? 4 * (size_t)CROSS_TI * CROSS_CP : 0);
}

}  // namespace tqc
