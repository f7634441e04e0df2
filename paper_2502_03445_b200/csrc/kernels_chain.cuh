// Fused small-bond chain (sm_100a): when every per-state step of a plan is small, the whole per-state tail of the
// contraction tree — gathers (a3), pairwise contractions (a4) and the final reduction (a5) —
// runs in ONE kernel, one warp per state, with every intermediate kept in that warp's shared memory instead of
// round-tripping through HBM.  Bond sums that have fewer than 32 outputs are split over lanes and finished with warp
// shuffles.  The step table is plan data (built once on the host, read from global memory).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "device_args.h"

namespace tqc {

constexpr int CHAIN_MAX_STEPS = 24;
constexpr int CHAIN_WARPS = 8;                 // warps (states in flight) per block

struct ChainOperand {
    const float *base;       // LEAF: its device tensor (rows of 2^{lgRows+lgK} floats)
    long long table_ofs;     // TABLE: float offset inside the workspace's table region (-1 otherwise)
    int gathered;            // 1: LEAF or TABLE row selected by the state's key; 0: intermediate in shared memory
    int key_slot;            // gathered: row = keys[key_slot * cap + r]
    int smem_ofs;            // float offset in the warp's scratch: staging area (gathered, staged) or the intermediate itself
    int staged;              // gathered operand copied to shared memory first (it is reused by several outputs)
    int pitch;               // floats between consecutive rows where the inner loop reads it (K, or K + 4 in shared memory)
};

struct ChainStep {
    ChainOperand A, B;
    int lgM, lgN, lgK;
    int c_smem_ofs;          // result: float offset in the warp's scratch, or -1: the root, written to out[r]
    int c_lgK;               // log2 of the row length the consumer reads the result with (rows are padded by 4 floats)
    BitMap outA, outB;       // i -> bits of the result's linear index, j -> bits (disjoint)
};

struct ChainArgs {
    const ChainStep *steps;  // DEVICE [n_steps]
    int n_steps;
    const float *tables;     // states-mode table region of the workspace
    const uint32_t *keys;    // [n_slots][cap]
    long long cap;
    float *out;
    int R;
    int scratch_floats;      // per warp
};

// index of element x of a padded intermediate: rows of 2^lgK floats, 4 floats of padding per row (bank spread for float4 reads)
__device__ __forceinline__ int chain_pad(int x, int lgK) { return lgK >= 2 ? x + ((x >> lgK) << 2) : x; }

__device__ __forceinline__ float dot_range(const float *pa, const float *pb, int k_lo, int k_hi) {
    float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
    if (k_hi - k_lo >= 4) {
        for (int k = k_lo; k < k_hi; k += 4) {
            const float4 x = *reinterpret_cast<const float4 *>(pa + k), y = *reinterpret_cast<const float4 *>(pb + k);
            s0 = fmaf(x.x, y.x, s0); s1 = fmaf(x.y, y.y, s1); s2 = fmaf(x.z, y.z, s2); s3 = fmaf(x.w, y.w, s3);
        }
    } else {
        for (int k = k_lo; k < k_hi; ++k) s0 = fmaf(pa[k], pb[k], s0);
    }
    return (s0 + s1) + (s2 + s3);
}

__global__ void __launch_bounds__(CHAIN_WARPS * 32) chain_kernel(const ChainArgs a) {
    extern __shared__ __align__(16) float chain_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float *scr = chain_smem + (size_t)warp * a.scratch_floats;
    const long long n_warps = (long long)gridDim.x * CHAIN_WARPS;
    for (long long r = (long long)blockIdx.x * CHAIN_WARPS + warp; r < a.R; r += n_warps) {
        for (int t = 0; t < a.n_steps; ++t) {
            const ChainStep &s = a.steps[t];
            const int M = 1 << s.lgM, N = 1 << s.lgN, K = 1 << s.lgK;
            // ---- operands: shared-memory intermediate, staged gather, or direct gather ----
            const float *pa, *pb;
            {
                const ChainOperand &o = s.A;
                if (!o.gathered) pa = scr + o.smem_ofs;
                else {
                    const float *g = (o.table_ofs >= 0 ? a.tables + o.table_ofs : o.base) +
                                     ((size_t)a.keys[(long long)o.key_slot * a.cap + r] << (s.lgM + s.lgK));
                    if (o.staged) {
                        float *d = scr + o.smem_ofs;
                        for (int x = lane * 4; x < M * K; x += 128)
                            *reinterpret_cast<float4 *>(d + chain_pad(x, s.lgK)) = __ldg(reinterpret_cast<const float4 *>(g + x));
                        pa = d;
                    } else pa = g;
                }
            }
            {
                const ChainOperand &o = s.B;
                if (!o.gathered) pb = scr + o.smem_ofs;
                else {
                    const float *g = (o.table_ofs >= 0 ? a.tables + o.table_ofs : o.base) +
                                     ((size_t)a.keys[(long long)o.key_slot * a.cap + r] << (s.lgN + s.lgK));
                    if (o.staged) {
                        float *d = scr + o.smem_ofs;
                        for (int x = lane * 4; x < N * K; x += 128)
                            *reinterpret_cast<float4 *>(d + chain_pad(x, s.lgK)) = __ldg(reinterpret_cast<const float4 *>(g + x));
                        pb = d;
                    } else pb = g;
                }
            }
            __syncwarp();
            // ---- outputs: G lanes share one output when there are fewer than 32 of them ----
            const int lgO = s.lgM + s.lgN;
            int lgG = lgO >= 5 ? 0 : 5 - lgO;
            if (s.lgK - lgG < 2) lgG = s.lgK >= 2 ? s.lgK - 2 : 0;        // at least one float4 of k per lane
            const int G = 1 << lgG, kspan = K >> lgG;
            const int g = lane & (G - 1);
            const int per_pass = 32 >> lgG;
            for (int o0 = 0; o0 < (1 << lgO); o0 += per_pass) {
                const int o = o0 + (lane >> lgG);
                float v = 0.f;
                const bool live = o < (1 << lgO);
                const int i = o >> s.lgN, j = o & (N - 1);
                if (live) v = dot_range(pa + (size_t)i * s.A.pitch, pb + (size_t)j * s.B.pitch, g * kspan, (g + 1) * kspan);
                for (int d = G >> 1; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
                if (live && g == 0) {
                    if (s.c_smem_ofs < 0) a.out[r] = v;
                    else {
                        const int x = (int)(bitmap_apply(s.outA, (unsigned long long)i) | bitmap_apply(s.outB, (unsigned long long)j));
                        scr[s.c_smem_ofs + chain_pad(x, s.c_lgK)] = v;
                    }
                }
            }
            __syncwarp();
        }
    }
}

}  // namespace tqc
