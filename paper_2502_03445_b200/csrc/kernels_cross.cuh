// Table steps with a short bond (K = 8 .. 64) and many rows on both sides: the cross-mode contraction of a4/a6
//     C[outA(i') | outB(j')] = sum_k A[rowA(i'), k] * B[rowB(j'), k]
// is one M' x N' x K product per step (PAPER.md lines 318-330 merged bond).  With K this
// short the fp32 FFMA kernel is bound by instruction issue, not by the result write, so the products run on the tensor
// pipe as warp-level 3xTF32 mma.sync blocks (kernels_chain.cuh: chain_step_mma, one bond slice of 8 per accumulator and the
// slices added in registers: table steps feed one another and the pipe's truncating accumulator would drift), 64 x 128
// outputs per 256-thread block.
// Where j' and j' + 1 are neighbours in C (the usual case: the result layout keeps the operand's digit order) the results
// leave straight from the fragments as 16-byte stores after a lane exchange, 64 contiguous bytes per quad; otherwise the tile goes through
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
        // results leave straight from the fragments, no trip through shared memory
        // (columns j .. j + 3, j a multiple of 4, are neighbours in C: neighbouring lanes of a quad swap halves of two 8-column
        // fragments, an even lane then holds 4 consecutive columns of fragment 2 n, the odd lane next to it 4 of fragment
        // 2 n + 1, and a lane stores 16 bytes - a quad writes 64 contiguous bytes of a row: kernels_tc2.cuh, store-path numbers
        // in DESIGN.md 5.2)
        const int wi = warp >> 2, wj = warp & 3;
        const int g = lane >> 2, t = lane & 3;
        const bool odd = (t & 1) != 0;
        float acc[2][4][4];
        chain_mma_acc<5, 5, LGK, P, P, true>(As + 32 * wi * P, Bs + 32 * wj * P, lane, acc);
#pragma unroll
        for (int mi = 0; mi < 2; ++mi)
#pragma unroll
            for (int np = 0; np < 2; ++np) {
                const float *e = acc[mi][2 * np], *o = acc[mi][2 * np + 1];
                const float r0 = __shfl_xor_sync(0xffffffffu, odd ? e[0] : o[0], 1), r1 = __shfl_xor_sync(0xffffffffu, odd ? e[1] : o[1], 1);
                const float r2 = __shfl_xor_sync(0xffffffffu, odd ? e[2] : o[2], 1), r3 = __shfl_xor_sync(0xffffffffu, odd ? e[3] : o[3], 1);
                const unsigned long long ob = offB[32 * wj + 8 * (2 * np + (odd ? 1 : 0)) + 2 * (t & 2)];
                float *ctop = a.C + (offA[32 * wi + 16 * mi + g] | ob), *cbot = a.C + (offA[32 * wi + 16 * mi + g + 8] | ob);
                *reinterpret_cast<float4 *>(ctop) = odd ? make_float4(r0, r1, o[0], o[1]) : make_float4(e[0], e[1], r0, r1);
                *reinterpret_cast<float4 *>(cbot) = odd ? make_float4(r2, r3, o[2], o[3]) : make_float4(e[2], e[3], r2, r3);
            }
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
