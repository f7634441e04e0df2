// kernels_sim.cuh — batched statevector simulation of the subcircuit variants and the Pauli attribution that turns
// them into the subcircuit tensor T_s (section 2.1).
//
// A subcircuit with d downstream cut wires and u upstream cut wires has 4^d * 3^u variants: every downstream wire is
// initialised in one of |0>, |1>, |+>, |i> and every upstream wire is measured in Z, X or Y ("only 3 ... per upstream
// cut": I and Z share the Z setting).  The variants of one preparation differ only in the
// measurement rotations, so a thread block simulates one preparation once - the 2^w complex128 amplitudes live in
// shared memory for the whole run (w <= 13: 192 KB with the probabilities), every gate is one pass over them - and
// then walks a share of the 3^u settings; per setting: the rotation, |amp|^2, a Walsh-Hadamard pass over the upstream
// wires that forms the signed sums over the measured bits for every basis at once, and a scatter of the
// 2^{#Z settings} * 2^o results into R[a][k_u][x].  The downstream bases are then "constructed as a linear combination from the initialization states"
// (line 188; coefficients: DESIGN.md reading G3) one axis at a time, and the result is written in the caller's axis
// order as fp32.  All arithmetic is fp64 (B200 has full-rate FP64 units; the work is tiny next to the contraction).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace tqc {

struct SimGate {
    int32_t nq;        // 1 or 2 operands
    int32_t b0, b1;    // bit position (in the amplitude index) of the first / second operand; first = more significant
    int32_t pad;
    double2 m[16];     // row-major 2x2 or 4x4 unitary, m[r * dim + c]
};

struct SimArgs {
    int32_t w, d, u, o, n_gates;
    int32_t g;                                 // the first g upstream wires' settings come from blockIdx, the rest are walked
    int32_t D_bit[16], U_bit[16], O_bit[32];   // amplitude-index bit positions of the listed wires
    const SimGate *gates;
    double *R;                                 // [4^d][4^u][2^o]
    double2 *scratch;                          // w >= 14 only: per block 2^w complex128 amplitudes + 2^w float64 probabilities
};

__device__ __forceinline__ double2 cfma(double2 a, double2 b, double2 acc) {
    acc.x += a.x * b.x - a.y * b.y;
    acc.y += a.x * b.y + a.y * b.x;
    return acc;
}

__device__ __forceinline__ uint32_t insert_zero(uint32_t p, int bit) {
    return ((p >> bit) << (bit + 1)) | (p & ((1u << bit) - 1u));
}

__device__ __forceinline__ void sim_apply_1q(double2 *psi, int w, int bit, const double2 *m) {
    const double2 m00 = m[0], m01 = m[1], m10 = m[2], m11 = m[3];
    for (uint32_t p = threadIdx.x; p < (1u << (w - 1)); p += blockDim.x) {
        const uint32_t i0 = insert_zero(p, bit), i1 = i0 | (1u << bit);
        const double2 a0 = psi[i0], a1 = psi[i1];
        psi[i0] = cfma(m01, a1, cfma(m00, a0, make_double2(0.0, 0.0)));
        psi[i1] = cfma(m11, a1, cfma(m10, a0, make_double2(0.0, 0.0)));
    }
    __syncthreads();
}

__device__ __forceinline__ void sim_apply_2q(double2 *psi, int w, int b0, int b1, const double2 *m) {
    const int lo = b0 < b1 ? b0 : b1, hi = b0 < b1 ? b1 : b0;
    for (uint32_t p = threadIdx.x; p < (1u << (w - 2)); p += blockDim.x) {
        const uint32_t base = insert_zero(insert_zero(p, lo), hi);
        uint32_t idx[4];
        double2 v[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            idx[c] = base | (uint32_t(c >> 1) << b0) | (uint32_t(c & 1) << b1);
            v[c] = psi[idx[c]];
        }
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            double2 acc = make_double2(0.0, 0.0);
#pragma unroll
            for (int c = 0; c < 4; ++c) acc = cfma(m[r * 4 + c], v[c], acc);
            psi[idx[r]] = acc;
        }
    }
    __syncthreads();
}

// Reflected ternary Gray code: digit k (0 = least significant) of step t.  Consecutive steps differ in one digit by +-1.
__device__ __forceinline__ int gray3_digit(uint32_t t, uint32_t pow3k) {
    const uint32_t q = t / pow3k;
    const int dgt = int(q % 3);
    return ((q / 3) & 1u) ? 2 - dgt : dgt;
}

// blockIdx.x = a * 3^g + group.  a in base 4 (first downstream wire = most significant digit, 0..3 = |0>,|1>,|+>,|i>).
// The block simulates preparation a ONCE and then walks 3^{u-g} measurement settings (0..2 = Z, X, Y): the settings of
// the first g upstream wires are the base-3 digits of `group`, those of the other u-g wires run through a reflected
// Gray code, so going from one setting to the next is ONE one-qubit pass (new rotation times the inverse of the old one).
// Shared memory: 2^w complex128 amplitudes followed by 2^w float64 probabilities (w <= 13: 192 KB).  IN_GLOBAL: subcircuits of
// 14 and 15 wires (the paper's cap) keep the same 24 * 2^w bytes per block in the caller's workspace,
// where they stay L2-resident (at most 2 * 148 blocks x 768 KB); the passes are the same code on a global pointer.
template <bool IN_GLOBAL>
__global__ void __launch_bounds__(512) sim_variant_kernel(SimArgs g) {
    extern __shared__ double2 psi_smem[];
    __shared__ double2 rot[4][4];
    const int w = g.w, u = g.u, ng = g.g;
    const uint32_t size = 1u << w;
    double2 *psi = IN_GLOBAL ? g.scratch + (size_t)blockIdx.x * (size + size / 2) : psi_smem;
    double *q = reinterpret_cast<double *>(psi + size);
    uint32_t pow3g = 1, n_walk = 1;
    for (int j = 0; j < ng; ++j) pow3g *= 3;
    for (int j = ng; j < u; ++j) n_walk *= 3;
    const uint32_t a = blockIdx.x / pow3g, group = blockIdx.x % pow3g;
    const double r = 0.70710678118654752440;

    // initial product state: downstream wires prepared, every other wire in |0>
    uint32_t dmask = 0;
    for (int i = 0; i < g.d; ++i) dmask |= 1u << g.D_bit[i];
    for (uint32_t idx = threadIdx.x; idx < size; idx += blockDim.x) {
        double2 amp = make_double2((idx & ~dmask) ? 0.0 : 1.0, 0.0);
        for (int i = 0; i < g.d; ++i) {
            const int ai = (a >> (2 * (g.d - 1 - i))) & 3, bit = (idx >> g.D_bit[i]) & 1;
            double2 f;
            if (ai == 0) f = make_double2(bit ? 0.0 : 1.0, 0.0);
            else if (ai == 1) f = make_double2(bit ? 1.0 : 0.0, 0.0);
            else if (ai == 2) f = make_double2(r, 0.0);
            else f = bit ? make_double2(0.0, r) : make_double2(r, 0.0);
            amp = cfma(amp, f, make_double2(0.0, 0.0));
        }
        psi[idx] = amp;
    }
    if (threadIdx.x == 0) {
        // rotate so that a Z measurement reads the basis.  rot[0]: X setting, H (also Z -> X and X -> Z: H is its own
        // inverse).  rot[1]: Y setting, H Sdg = [[1, -i], [1, i]] / sqrt2.  rot[2]: X -> Y, (H Sdg) H.  rot[3]: Y -> X,
        // H (S H) = H (H Sdg)^-1.
        rot[0][0] = make_double2(r, 0.0); rot[0][1] = make_double2(r, 0.0);
        rot[0][2] = make_double2(r, 0.0); rot[0][3] = make_double2(-r, 0.0);
        rot[1][0] = make_double2(r, 0.0); rot[1][1] = make_double2(0.0, -r);
        rot[1][2] = make_double2(r, 0.0); rot[1][3] = make_double2(0.0, r);
        rot[2][0] = make_double2(0.5, -0.5); rot[2][1] = make_double2(0.5, 0.5);
        rot[2][2] = make_double2(0.5, 0.5); rot[2][3] = make_double2(0.5, -0.5);
        rot[3][0] = make_double2(0.5, 0.5); rot[3][1] = make_double2(0.5, -0.5);
        rot[3][2] = make_double2(0.5, -0.5); rot[3][3] = make_double2(0.5, 0.5);
    }
    __syncthreads();

    for (int t = 0; t < g.n_gates; ++t) {
        const SimGate *gt = g.gates + t;
        if (gt->nq == 1) sim_apply_1q(psi, w, gt->b0, gt->m);
        else sim_apply_2q(psi, w, gt->b0, gt->b1, gt->m);
    }

    // settings of the fixed wires (the walked wires start at Z: no rotation)
    {
        uint32_t rem = group;
        for (int j = ng - 1; j >= 0; --j) {
            const int bj = rem % 3;
            rem /= 3;
            if (bj) sim_apply_1q(psi, w, g.U_bit[j], rot[bj - 1]);
        }
    }
    for (uint32_t step = 0; step < n_walk; ++step) {
        // q[x_O, b_U] = |amp|^2
        for (uint32_t idx = threadIdx.x; idx < size; idx += blockDim.x) {
            const double2 v = psi[idx];
            q[idx] = v.x * v.x + v.y * v.y;
        }
        __syncthreads();
        // signed sums over the measured bits: sigma(I, b) = +1, sigma(X|Y|Z, b) = (-1)^b.  After the pass, the entry whose
        // upstream bit is 0 holds the I sum and the entry whose bit is 1 holds the signed sum.
        for (int j = 0; j < u; ++j) {
            const int bit = g.U_bit[j];
            for (uint32_t p = threadIdx.x; p < (size >> 1); p += blockDim.x) {
                const uint32_t i0 = insert_zero(p, bit), i1 = i0 | (1u << bit);
                const double p0 = q[i0], p1 = q[i1];
                q[i0] = p0 + p1;
                q[i1] = p0 - p1;
            }
            __syncthreads();
        }
        // scatter: a Z setting serves I (bit 0) and Z (bit 1); an X or Y setting serves only its own basis (bit 1)
        for (uint32_t idx = threadIdx.x; idx < size; idx += blockDim.x) {
            uint32_t ku = 0, rem = group, pw = 1;
            bool keep = true;
            for (int j = u - 1; j >= 0; --j) {
                int bj;
                if (j >= ng) { bj = gray3_digit(step, pw); pw *= 3; }
                else { bj = rem % 3; rem /= 3; }
                const int bit = (idx >> g.U_bit[j]) & 1;
                const uint32_t digit = bj == 0 ? (bit ? 3u : 0u) : uint32_t(bj);
                keep = keep && (bj == 0 || bit);
                ku |= digit << (2 * (u - 1 - j));
            }
            if (!keep) continue;
            uint32_t x = 0;
            for (int j = 0; j < g.o; ++j) x = (x << 1) | ((idx >> g.O_bit[j]) & 1u);
            g.R[((((size_t(a) << (2 * u)) + ku)) << g.o) + x] = q[idx];
        }
        // next setting: the one walked wire whose Gray digit changes
        if (step + 1 < n_walk) {
            uint32_t pw = 1;
            for (int j = u - 1; j >= ng; --j, pw *= 3) {
                const int from = gray3_digit(step, pw), to = gray3_digit(step + 1, pw);
                if (from == to) continue;
                // 0 <-> 1: H;  1 -> 2: (H Sdg) H;  2 -> 1: H (S H)
                const int which = (from + to == 1) ? 0 : (to == 2 ? 2 : 3);
                sim_apply_1q(psi, w, g.U_bit[j], rot[which]);     // ends with __syncthreads (also fences the scatter reads)
            }
        }
    }
}

// Downstream linear combination along one prep axis, in place.  R is [outer][4][inner]; rows over (|0>,|1>,|+>,|i>):
// I = (1, 1, 0, 0), X = (-1, -1, 2, 0), Y = (-1, -1, 0, 2), Z = (1, -1, 0, 0)  (reading G3).
__global__ void sim_kappa_axis_kernel(double *R, size_t inner, size_t n_tuples) {
    for (size_t t = size_t(blockIdx.x) * blockDim.x + threadIdx.x; t < n_tuples; t += size_t(gridDim.x) * blockDim.x) {
        const size_t outer = t / inner, in = t - outer * inner;
        double *p = R + outer * 4 * inner + in;
        const double r0 = p[0], r1 = p[inner], r2 = p[2 * inner], r3 = p[3 * inner];
        const double s = r0 + r1;
        p[0] = s;
        p[inner] = 2.0 * r2 - s;
        p[2 * inner] = 2.0 * r3 - s;
        p[3 * inner] = r0 - r1;
    }
}

struct SimPermArgs {
    int32_t c, o;
    int32_t pos[32];   // bond j of R's order (downstream wires first, then upstream) -> digit position in the output row
};

// out[row'(digits)][x] = (float) R[row][x]: the caller's axis order (tqc.h: first listed incident cut = most significant).
__global__ void sim_permute_cast_kernel(const double *R, float *out, SimPermArgs g, size_t total) {
    for (size_t t = size_t(blockIdx.x) * blockDim.x + threadIdx.x; t < total; t += size_t(gridDim.x) * blockDim.x) {
        const size_t row = t >> g.o, x = t & ((size_t(1) << g.o) - 1);
        size_t orow = 0;
        for (int j = 0; j < g.c; ++j) {
            const size_t digit = (row >> (2 * (g.c - 1 - j))) & 3;
            orow |= digit << (2 * (g.c - 1 - g.pos[j]));
        }
        out[(orow << g.o) + x] = float(R[t]);
    }
}

}  // namespace tqc
