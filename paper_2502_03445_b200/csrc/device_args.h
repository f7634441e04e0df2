// Kernel argument structures shared by the host launchers (tqc_api.cu) and the kernels.
// Every dimension on the path is a power of two (a cut bond has 4 values, an output qubit 2), so
// all index arithmetic is bit routing: a BitMap sends runs of source index bits to destination
// bit positions.  It expresses, with one mechanism,
//   - the digit permutation between the caller's tensor axes and the device layout (a1, G6),
//   - the scatter of a contraction result into the digit order its consumer wants (a4),
//   - the deposit of free output bits around a fixed prefix (a6), and
//   - the product-order -> global-bit-order permutation of the distribution (a6, G4).
#pragma once
#if defined(__CUDACC_RTC__)      // run-time compilation (chain_jit.cpp): no standard headers
typedef unsigned char uint8_t;
typedef unsigned short uint16_t;
typedef int int32_t;
typedef unsigned int uint32_t;
typedef unsigned long long uint64_t;
#else
#include <stdint.h>
#endif

#define TQC_MAXSEG 48

struct BitMap {                 // y = OR_s (((x >> src[s]) & ((1 << len[s]) - 1)) << dst[s])
    int32_t n;
    uint8_t src[TQC_MAXSEG], len[TQC_MAXSEG], dst[TQC_MAXSEG];
};

#if defined(__CUDACC__)
__host__ __device__
#endif
static inline unsigned long long bitmap_apply(const BitMap &m, unsigned long long x) {
    unsigned long long y = 0;
    for (int s = 0; s < m.n; ++s)
        y |= ((x >> m.src[s]) & ((1ull << m.len[s]) - 1ull)) << m.dst[s];
    return y;
}

// One operand of a contraction step, seen as a K-major matrix.
//   batch mode: element (r, i, k) = base[(row(r) * rows_inner + i) * K + k], row(r) = keys ? keys[r] : r
//   cross mode: element (i', k)   = base[((in_map(i') | in_or)) * K + k]   (i' = table-row bits ++ digits)
struct OperandArgs {
    const float *base;
    const uint32_t *keys;
    BitMap in_map;
    unsigned long long in_or;
    int use_map;                // cross mode with a non-identity row mapping (leaf under a prefix)
};

struct StepArgs {
    OperandArgs A, B;
    float *C;
    BitMap outA, outB;          // i' -> bits of the C offset, j' -> bits of the C offset (disjoint)
    long long c_row_stride;     // batch mode: floats per row of C (4^{#open cuts of C})
    int lgM, lgN, lgK;          // log2 of the virtual dimensions M' x N' x K (batch mode: per row)
    int R;                      // rows (states of the chunk) in batch mode; 1 in cross mode
    int lgTI, lgTJ, lgTK, lgRPB;        // log2 of the tile of one block: RPB rows x TI x TJ outputs, K in slabs of TK
    int lgTilesI, lgTilesJ;             // log2 of the tile counts M / TI, N / TJ
    int vec_store;              // the 4 consecutive j of a thread are contiguous in C
};

struct DotArgs {                // a5: out[r] = sum_k A_r[k] * B_r[k]
    const float *A, *B;
    const uint32_t *keysA, *keysB;
    float *out;
    int lgK, R;
};

struct KeyArgs {                // a2: keys[slot][r] = packed output bits of the slot's node
    const uint64_t *states;     // [R][words]
    uint32_t *keys;             // [n_slots][cap]
    const int32_t *slot_ofs;    // [n_slots + 1]
    const int32_t *slot_qubits; // qubits of each slot, first = MSB
    int words, R;
    long long cap;
};

struct RelayoutArgs {           // a1: dst[x][j] = scale * src[row_of(j)][x]
    const float *src;
    float *dst;
    BitMap row_of;              // device digit index j -> caller row index
    unsigned long long row_or;  // fixed digits of the caller row index (sliced axes), 0 without slicing
    int lgRows, lgCols;         // caller layout: 2^lgRows rows (4^{c_s}) x 2^lgCols columns (2^{o_s})
    float scale;                // exact power of two 2^{-d_s}
};

struct GatherArgs {             // out[r] = table[keys ? keys[r] : (map(r) | or)]   (root is a LEAF or TABLE)
    const float *table;
    const uint32_t *keys;
    BitMap map;
    unsigned long long map_or;
    BitMap out_map;             // distribution: row r -> out index
    float *out;
    long long R;
};
