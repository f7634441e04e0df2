// SIMT kernels of the reconstruction hot path (sm_100a).  PAPER.md section 3.2 (lines 321-330):
// a pairwise contraction multiplies two tensors and sums over their shared (merged) bond;
// section 3.3 (lines 407-412): it costs 4^{#inner + #outer} multiplications per state.
#pragma once
#include <cuda_runtime.h>
#include "device_args.h"

namespace tqc {

// ---------------------------------------------------------------------------------------------
// a1  load / re-layout:  dst[x][j] = scale * src[row_of(j)][x]
// 32x32 shared-memory transpose: reads run along x (contiguous in the caller's layout), writes
// along j (contiguous in the state-major device layout).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) relayout_kernel(const RelayoutArgs a) {
    __shared__ float tile[32][33];
    const long long rows = 1ll << a.lgRows, cols = 1ll << a.lgCols;
    const long long tiles_x = (cols + 31) / 32;
    const long long bx = blockIdx.x % tiles_x, bj = blockIdx.x / tiles_x;
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const long long x = bx * 32 + tx;
    for (int jj = ty; jj < 32; jj += 8) {
        const long long j = bj * 32 + jj;
        if (j < rows && x < cols) {
            const unsigned long long row = bitmap_apply(a.row_of, (unsigned long long)j) | a.row_or;
            tile[jj][tx] = a.src[row * cols + x];
        }
    }
    __syncthreads();
    const long long j = bj * 32 + tx;
    for (int xx = ty; xx < 32; xx += 8) {
        const long long xo = bx * 32 + xx;
        if (j < rows && xo < cols) a.dst[xo * rows + j] = a.scale * tile[tx][xx];
    }
}

// ---------------------------------------------------------------------------------------------
// a2  key extraction:  keys[slot][r] = bits of state r at the slot's qubits, first listed = MSB
// (readings G4, G5: qubit q is bit q%64 of word q/64).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) key_kernel(const KeyArgs a) {
    const int slot = blockIdx.y;
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= a.R) return;
    const uint64_t *w = a.states + r * a.words;
    uint32_t key = 0;
    for (int p = a.slot_ofs[slot]; p < a.slot_ofs[slot + 1]; ++p) {
        const int q = a.slot_qubits[p];
        key = (key << 1) | (uint32_t)((w[q >> 6] >> (q & 63)) & 1ull);
    }
    a.keys[slot * a.cap + r] = key;
}

// ---------------------------------------------------------------------------------------------
// a3 + a4  contraction step, register-tiled fp32 FFMA.
//   C[rowC][outA(i') | outB(j')] = sum_k A[i', k] * B[j', k]
// Both operands are K-major (the merged bond is the contiguous axis).  The gather of a3 is the
// operand addressing: a row of a LEAF/TABLE operand is selected by the state's key.
// One block: RPB rows x (TI x TJ) outputs; each thread an MI x MJ micro-tile; the bond is
// consumed in slabs of TK staged through shared memory as [k][i] so the inner loop reads
// float4s that are broadcast (A) or contiguous (B) across a warp.
// ---------------------------------------------------------------------------------------------
template <int MI, int MJ>
__global__ void __launch_bounds__(256, 4) step_tile_kernel(const StepArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    // every tile dimension is a power of two: all index splitting below is shifts and masks
    constexpr int LGMI = MI == 4 ? 2 : 0, LGMJ = MJ == 4 ? 2 : 0;
    const int lgTI = a.lgTI, lgTJ = a.lgTJ, lgTK = a.lgTK;
    const int TI = 1 << lgTI, TJ = 1 << lgTJ, TK = 1 << lgTK, RPB = 1 << a.lgRPB;
    const int TIp = TI + (MI == 4 ? 4 : 1), TJp = TJ + (MJ == 4 ? 4 : 1);
    unsigned long long *rowA = reinterpret_cast<unsigned long long *>(smem_raw);     // [RPB*TI] float offsets
    unsigned long long *rowB = rowA + RPB * TI;                                       // [RPB*TJ]
    unsigned long long *offA = rowB + RPB * TJ;                                       // [TI] C offset bits of i'
    unsigned long long *offB = offA + TI;                                             // [TJ] C offset bits of j'
    float *As = reinterpret_cast<float *>(offB + TJ + ((RPB * (TI + TJ) + TI + TJ) & 1));   // [RPB][TK][TIp], 16 B aligned
    float *Bs = As + ((RPB * TK * TIp + 3) & ~3);                                     // [RPB][TK][TJp], 16 B aligned

    const long long bid = blockIdx.x;
    const int tjb = (int)(bid & ((1ll << a.lgTilesJ) - 1));
    const int tib = (int)((bid >> a.lgTilesJ) & ((1ll << a.lgTilesI) - 1));
    const long long rg = bid >> (a.lgTilesJ + a.lgTilesI);
    const int lg_ntj = lgTJ - LGMJ, lg_tpr = (lgTI - LGMI) + lg_ntj;
    const int tid = threadIdx.x;
    const int row_l = tid >> lg_tpr, within = tid & ((1 << lg_tpr) - 1);
    const int ti = within >> lg_ntj, tj = within & ((1 << lg_ntj) - 1);
    const long long K = 1ll << a.lgK;
    const long long M = 1ll << a.lgM, N = 1ll << a.lgN;

    // operand row offsets (in floats) of every (row, i) and (row, j) this block touches; C offset bits of i' and j'
    for (int e = tid; e < RPB * TI; e += 256) {
        const int rl = e >> lgTI, i = e & (TI - 1);
        const long long r = (rg << a.lgRPB) + rl;
        const unsigned long long ip = ((unsigned long long)tib << lgTI) + i;
        unsigned long long off = ~0ull;
        if (r < a.R) {
            if (a.A.use_map) off = (bitmap_apply(a.A.in_map, ip) | a.A.in_or) << a.lgK;
            else {
                const unsigned long long row = a.A.keys ? (unsigned long long)a.A.keys[r] : (unsigned long long)r;
                off = ((row << a.lgM) + ip) << a.lgK;
            }
        }
        rowA[e] = off;
        if (rl == 0) offA[i] = bitmap_apply(a.outA, ip);
    }
    for (int e = tid; e < RPB * TJ; e += 256) {
        const int rl = e >> lgTJ, j = e & (TJ - 1);
        const long long r = (rg << a.lgRPB) + rl;
        const unsigned long long jp = ((unsigned long long)tjb << lgTJ) + j;
        unsigned long long off = ~0ull;
        if (r < a.R) {
            if (a.B.use_map) off = (bitmap_apply(a.B.in_map, jp) | a.B.in_or) << a.lgK;
            else {
                const unsigned long long row = a.B.keys ? (unsigned long long)a.B.keys[r] : (unsigned long long)r;
                off = ((row << a.lgN) + jp) << a.lgK;
            }
        }
        rowB[e] = off;
        if (rl == 0) offB[j] = bitmap_apply(a.outB, jp);
    }
    __syncthreads();

    float acc[MI][MJ];
#pragma unroll
    for (int x = 0; x < MI; ++x)
#pragma unroll
        for (int y = 0; y < MJ; ++y) acc[x][y] = 0.f;

    for (long long k0 = 0; k0 < K; k0 += TK) {
        if (lgTK >= 2) {
            const int lgkq = lgTK - 2;
            for (int e = tid; e < (RPB << (lgTI + lgkq)); e += 256) {
                const int k4 = e & ((1 << lgkq) - 1), ri = e >> lgkq;          // ri = rl * TI + i
                const unsigned long long off = rowA[ri];
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (off != ~0ull) v = __ldg(reinterpret_cast<const float4 *>(a.A.base + off + k0) + k4);
                float *dst = As + (((ri >> lgTI) << lgTK) + k4 * 4) * TIp + (ri & (TI - 1));
                dst[0] = v.x; dst[TIp] = v.y; dst[2 * TIp] = v.z; dst[3 * TIp] = v.w;
            }
            for (int e = tid; e < (RPB << (lgTJ + lgkq)); e += 256) {
                const int k4 = e & ((1 << lgkq) - 1), rj = e >> lgkq;
                const unsigned long long off = rowB[rj];
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (off != ~0ull) v = __ldg(reinterpret_cast<const float4 *>(a.B.base + off + k0) + k4);
                float *dst = Bs + (((rj >> lgTJ) << lgTK) + k4 * 4) * TJp + (rj & (TJ - 1));
                dst[0] = v.x; dst[TJp] = v.y; dst[2 * TJp] = v.z; dst[3 * TJp] = v.w;
            }
        } else {
            for (int e = tid; e < (RPB << (lgTI + lgTK)); e += 256) {
                const int k = e & (TK - 1), ri = e >> lgTK;
                const unsigned long long off = rowA[ri];
                As[(((ri >> lgTI) << lgTK) + k) * TIp + (ri & (TI - 1))] = (off != ~0ull) ? __ldg(a.A.base + off + k0 + k) : 0.f;
            }
            for (int e = tid; e < (RPB << (lgTJ + lgTK)); e += 256) {
                const int k = e & (TK - 1), rj = e >> lgTK;
                const unsigned long long off = rowB[rj];
                Bs[(((rj >> lgTJ) << lgTK) + k) * TJp + (rj & (TJ - 1))] = (off != ~0ull) ? __ldg(a.B.base + off + k0 + k) : 0.f;
            }
        }
        __syncthreads();
        if (row_l < RPB) {
            const float *ap = As + (row_l << lgTK) * TIp + ti * MI;
            const float *bp = Bs + (row_l << lgTK) * TJp + tj * MJ;
#pragma unroll 4
            for (int k = 0; k < TK; ++k) {
                float av[MI], bv[MJ];
                if (MI == 4) { const float4 t = *reinterpret_cast<const float4 *>(ap + k * TIp); av[0] = t.x; av[1] = t.y; av[2] = t.z; av[3] = t.w; }
                else av[0] = ap[k * TIp];
                if (MJ == 4) { const float4 t = *reinterpret_cast<const float4 *>(bp + k * TJp); bv[0] = t.x; bv[1] = t.y; bv[2] = t.z; bv[3] = t.w; }
                else bv[0] = bp[k * TJp];
#pragma unroll
                for (int x = 0; x < MI; ++x)
#pragma unroll
                    for (int y = 0; y < MJ; ++y) acc[x][y] = fmaf(av[x], bv[y], acc[x][y]);
            }
        }
        __syncthreads();
    }

    const long long r = (rg << a.lgRPB) + row_l;
    if (row_l >= RPB || r >= a.R) return;
    const unsigned long long i0 = ((unsigned long long)tib << lgTI) + ti * MI;
    const unsigned long long j0 = ((unsigned long long)tjb << lgTJ) + tj * MJ;
    if (i0 >= (unsigned long long)M || j0 >= (unsigned long long)N) return;
    float *crow = a.C + r * a.c_row_stride;
    unsigned long long ob[MJ];
#pragma unroll
    for (int y = 0; y < MJ; ++y) ob[y] = offB[tj * MJ + y];
#pragma unroll
    for (int x = 0; x < MI; ++x) {
        const unsigned long long oa = offA[ti * MI + x];
        if (MJ == 4 && a.vec_store) {
            *reinterpret_cast<float4 *>(crow + (oa | ob[0])) = make_float4(acc[x][0], acc[x][1], acc[x][2], acc[x][3]);
        } else {
#pragma unroll
            for (int y = 0; y < MJ; ++y) crow[oa | ob[y]] = acc[x][y];
        }
    }
}

// ---------------------------------------------------------------------------------------------
// a5  final reduction: no outer cut is left, out[r] = sum_k A_r[k] * B_r[k] over the last merged
// bond (the 2^{-K} of reading G1 is already folded into the leaves as 2^{-d_s}, reading G2).
// G lanes per row (G = min(32, K/4), float4 loads), shuffle tree inside the group.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) dot_kernel(const DotArgs a) {
    const long long K = 1ll << a.lgK;
    int G = (int)(K / 4);
    if (G > 32) G = 32;
    if (G < 1) G = 1;
    const int rows_per_warp = 32 / G;
    const int lane = threadIdx.x & 31;
    const long long warp = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long r = warp * rows_per_warp + lane / G;
    const int g = lane % G;
    float s = 0.f;
    if (r < a.R) {
        const unsigned long long ra = a.keysA ? (unsigned long long)a.keysA[r] : (unsigned long long)r;
        const unsigned long long rb = a.keysB ? (unsigned long long)a.keysB[r] : (unsigned long long)r;
        const float *pa = a.A + (ra << a.lgK), *pb = a.B + (rb << a.lgK);
        if (K >= 4) {
            const float4 *qa = reinterpret_cast<const float4 *>(pa), *qb = reinterpret_cast<const float4 *>(pb);
            float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
            for (long long k = g; k < K / 4; k += G) {
                const float4 x = __ldg(qa + k), y = __ldg(qb + k);
                s0 = fmaf(x.x, y.x, s0); s1 = fmaf(x.y, y.y, s1); s2 = fmaf(x.z, y.z, s2); s3 = fmaf(x.w, y.w, s3);
            }
            s = (s0 + s1) + (s2 + s3);
        } else {
            for (long long k = 0; k < K; ++k) s = fmaf(pa[k], pb[k], s);
        }
    }
    for (int d = G >> 1; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d, G);
    if (r < a.R && g == 0) a.out[r] = s;
}

// ---------------------------------------------------------------------------------------------
// root is a LEAF or a TABLE: out[...] = table[row]   (m = 1 / K = 0, or a network so small that
// the whole distribution is one table)
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) gather_kernel(const GatherArgs a) {
    const long long r = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= a.R) return;
    if (a.keys) a.out[r] = a.table[a.keys[r]];
    else a.out[bitmap_apply(a.out_map, (unsigned long long)r)] = a.table[bitmap_apply(a.map, (unsigned long long)r) | a.map_or];
}

// ---------------------------------------------------------------------------------------------
// Heavy State Selection, scoring pass (section 4, Alg. 1):
//   ||p_{j,i}|| = sqrt( sum_e (p_{j,i}^e)^2 )  for every binary state i of subcircuit j.
// In the state-major device layout state i is one contiguous row of 4^{c_j} floats, so the pass is a row norm: one warp
// per row, float4 loads, shuffle tree; HBM-bound (each tensor element read once).  `unscale` = 2^{d_j} undoes the exact
// power of two folded in at load, so the score is that of the caller's values.
// ---------------------------------------------------------------------------------------------
// out[i] += part[i]: the sum over sliced-bond sub-networks
__global__ void __launch_bounds__(256) accumulate_kernel(float *__restrict__ out, const float *__restrict__ part, long long n) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] += part[i];
}

template <int LANES>   // LANES = 32: one warp per row (many rows); LANES = 256: one block per row (few, long rows)
__global__ void __launch_bounds__(256) hss_norm_kernel(const float *__restrict__ t, float *__restrict__ score, long long rows,
                                                        int lgCols, float unscale) {
    __shared__ float part[8];
    const int lane = threadIdx.x & (LANES - 1);
    const long long group = LANES == 32 ? ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5 : blockIdx.x;
    const long long n_groups = LANES == 32 ? ((long long)gridDim.x * blockDim.x) >> 5 : gridDim.x;
    const long long cols = 1ll << lgCols;
    for (long long r = group; r < rows; r += n_groups) {
        const float *p = t + (r << lgCols);
        float s0 = 0.f, s1 = 0.f, s2 = 0.f, s3 = 0.f;
        if (cols >= 4) {
#pragma unroll 4
            for (long long k = lane * 4; k < cols; k += LANES * 4) {
                const float4 v = __ldg(reinterpret_cast<const float4 *>(p + k));
                s0 = fmaf(v.x, v.x, s0); s1 = fmaf(v.y, v.y, s1); s2 = fmaf(v.z, v.z, s2); s3 = fmaf(v.w, v.w, s3);
            }
        } else if (lane < cols) {
            s0 = p[lane] * p[lane];
        }
        float s = (s0 + s1) + (s2 + s3);
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (LANES == 256) {                              // fixed-order sum of the 8 warp partials
            if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = s;
            __syncthreads();
            s = ((part[0] + part[1]) + (part[2] + part[3])) + ((part[4] + part[5]) + (part[6] + part[7]));
            __syncthreads();
        }
        if (lane == 0) score[r] = sqrtf(s) * unscale;
    }
}

// ---------------------------------------------------------------------------------------------
// NEXT row 1, pruned output axes: the tensor of subcircuit j restricted to its heavy states x_j,
//     dst[i][q] = i < count ? src[keys[i]][perm(q)] : 0          i < 2^{ceil log2 count}
// a row gather on the state-major layout (rows are contiguous 4^{c} floats), with the digit order of the pruned plan.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) hss_rows_kernel(const float *__restrict__ src, float *__restrict__ dst,
                                                        const int32_t *__restrict__ keys, int count, long long rows_out,
                                                        int lgCols, const BitMap perm) {
    const long long n = rows_out << lgCols, stride = (long long)gridDim.x * blockDim.x;
    const long long cmask = (1ll << lgCols) - 1;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += stride) {
        const long long i = e >> lgCols;
        float v = 0.f;
        if (i < count) v = src[((long long)keys[i] << lgCols) + (long long)bitmap_apply(perm, (unsigned long long)(e & cmask))];
        dst[e] = v;
    }
}

struct HssCompactArgs {          // product order over the |x_j| (subcircuit 0 slowest) -> index in the padded 2^{v_j} table
    int m;
    int32_t count[64];
    uint8_t shift[64];
};
__global__ void __launch_bounds__(256) hss_compact_kernel(const float *__restrict__ padded, float *__restrict__ out, long long n,
                                                           const HssCompactArgs a) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long b = (long long)blockIdx.x * blockDim.x + threadIdx.x; b < n; b += stride) {
        long long rest = b;
        unsigned long long idx = 0;
        for (int j = a.m - 1; j >= 0; --j) {
            const long long cj = a.count[j];
            idx |= (unsigned long long)(rest % cj) << a.shift[j];
            rest /= cj;
        }
        out[b] = padded[idx];
    }
}

}  // namespace tqc
