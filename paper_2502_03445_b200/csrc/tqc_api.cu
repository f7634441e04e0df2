// C ABI of libtqc.so (include/tqc.h): plan handle, tensor load, states / distribution contraction.
// Host launch logic only; the arithmetic is in kernels_simt.cuh / kernels_tc.cuh.
#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <nvrtc.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/tqc.h"
#include "device_args.h"
#include "kernels_simt.cuh"
#include "kernels_tc.cuh"
#include "kernels_tc2.cuh"
#include "kernels_chain.cuh"
#include "kernels_cross.cuh"
#include "kernels_sim.cuh"
#include "plan.hpp"
#include "partition.hpp"

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg) {
    g_err = msg;
    return code;
}

#define TQC_CUDA(expr)                                                                         \
    do {                                                                                       \
        cudaError_t e__ = (expr);                                                              \
        if (e__ != cudaSuccess)                                                                \
            return fail(TQC_E_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e__));      \
    } while (0)

// ---- BitMap construction -------------------------------------------------------------------
struct BitPairs {
    std::vector<std::pair<int, int>> p;   // (src bit, dst bit)
    void add(int src, int dst) { p.emplace_back(src, dst); }
    void add_run(int src, int dst, int len) { for (int i = 0; i < len; ++i) add(src + i, dst + i); }
    bool build(BitMap &m) const {
        std::vector<std::pair<int, int>> q = p;
        std::sort(q.begin(), q.end());
        m.n = 0;
        for (size_t i = 0; i < q.size();) {
            size_t j = i + 1;
            while (j < q.size() && q[j].first == q[j - 1].first + 1 && q[j].second == q[j - 1].second + 1) ++j;
            if (m.n >= TQC_MAXSEG) return false;
            m.src[m.n] = (uint8_t)q[i].first; m.dst[m.n] = (uint8_t)q[i].second; m.len[m.n] = (uint8_t)(j - i);
            ++m.n;
            i = j;
        }
        return true;
    }
};

// Development switches (measurement variants of DESIGN.md 5.1).  A release build reads NO environment variable: the
// lookups below exist only when the library is compiled with -DTQC_DEVELOP (python -m paper_2502_03445_b200.build with
// TQC_DEVELOP=1 in the environment).
const char *dev_env(const char *name) {
#ifdef TQC_DEVELOP
    return std::getenv(name);
#else
    (void)name;
    return nullptr;
#endif
}

int index_of(const std::vector<int> &v, int x) {
    for (size_t i = 0; i < v.size(); ++i) if (v[i] == x) return (int)i;
    return -1;
}

}  // namespace

struct tqc_plan {
    tqc::HostPlan hp;
    tqc::PlanOptions plan_opts;
    int use_tcgen05 = 0;
    // fused small-bond chain (kernels_chain.cuh): the per-state steps as one device step table
    bool chain = false;
    std::vector<tqc::ChainStep> chain_host;
    std::vector<int> chain_leafA, chain_leafB;     // leaf id whose device pointer fills A.base / B.base (-1: none)
    tqc::ChainStep *d_chain = nullptr;
    std::vector<tqc::ChainGather> chain_gather;
    std::vector<int> chain_gather_leaf;
    int chain_scratch = 0, chain_stage = 0, chain_f4 = 0, chain_tab_entries = 0;
    // plan-specialised chain kernel, generated and compiled at the first contract call (chain_jit_build)
    int chain_mode = 0;                 // tqc_plan_opts.use_chain
    void *jit_module = nullptr, *jit_fn = nullptr;
    std::string jit_note;
    std::vector<float *> d_leaf;
    std::vector<char> loaded;
    int32_t *d_slot_ofs = nullptr, *d_slot_qubits = nullptr;
    float *d_staging = nullptr;
    size_t staging_elems = 0;
    uint64_t launches = 0, pair_launches = 0;      // all kernels / step_tc2_kernel (CTA-pair tensor-pipe steps)
    bool finalized = false;            // tqc_plan_finalize has run (device tables, specialised chain kernel, side streams)
    int sm_count = 0;
    // optional per-launch timing (tqc_plan_profile_*): one event before each launch + one at the end
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool;
    std::vector<int> ev_tags;          // tag of the launch that follows event i (same length as used events - 1)
    size_t ev_used = 0;
    // independent table steps run on side streams next to the key kernel (fork/join by events on the caller's stream)
    enum { N_LANES = 3 };
    cudaStream_t lane[N_LANES] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[N_LANES] = {nullptr, nullptr, nullptr};
    int tables_parallel = -1;          // -1 not decided; 0 serial; 1 fork/join
    // bond slicing: hp describes the network WITHOUT the sliced cuts; a leaf keeps one re-laid-out
    // sub-tensor per value of its sliced axes, the contract calls sum over all 4^{n_sliced} assignments
    int K_full = 0;
    std::vector<int> slice_cuts;                            // caller's cut ids; the first is the most significant digit
    std::vector<std::vector<int>> full_axis;                // per leaf: caller axis position (0 = MS) of every kept axis
    std::vector<std::vector<std::pair<int, int>>> sliced_axis;   // per leaf: (caller axis position, index into slice_cuts)
    std::vector<int> c_full, d_extra;                       // per leaf: caller's c_s; sliced cuts whose downstream end it holds
    std::vector<float *> d_leaf_all;                        // allocation per leaf: [4^{#sliced axes}][2^o][4^{c'}]
    int n_sliced() const { return (int)slice_cuts.size(); }
    // Heavy State Selection, pruned output axes: a distribution-mode plan of the same cut network whose subcircuit j
    // carries ceil(log2 |x_j|) virtual output bits (tqc_hss_prepare / tqc_hss_contract)
    tqc_plan *hss_sub = nullptr;
    std::vector<int32_t> hss_counts;
    // plans made by tqc_plan_from_circuit / _gates keep the cut description (partition, network, subcircuits)
    tqc::CutResult *cut = nullptr;
};

namespace {

using tqc::HostPlan;
using tqc::Node;
using tqc::Step;

constexpr int kMaxDynSmem = 200 * 1024;
constexpr int TQC_MAX_DEVICES = 64;

// Tags of profiled launches: step index t >= 0, or one of these.
enum { TAG_KEYS = -1, TAG_GATHER = -2, TAG_RELAYOUT = -3, TAG_CHAIN = -4, TAG_HSS = -5 };

int prof_event(tqc_plan_t *pl, cudaStream_t st) {
    if (pl->ev_used == pl->ev_pool.size()) {
        cudaEvent_t e;
        TQC_CUDA(cudaEventCreate(&e));
        pl->ev_pool.push_back(e);
    }
    TQC_CUDA(cudaEventRecord(pl->ev_pool[pl->ev_used++], st));
    return 0;
}
// called right before every kernel launch
int note_launch(tqc_plan_t *pl, int tag, cudaStream_t st) {
    pl->launches++;
    if (!pl->profile) return 0;
    pl->ev_tags.push_back(tag);
    return prof_event(pl, st);
}
int prof_begin(tqc_plan_t *pl) {
    if (pl->profile) { pl->ev_used = 0; pl->ev_tags.clear(); }
    return 0;
}
int prof_close(tqc_plan_t *pl, cudaStream_t st) { return pl->profile ? prof_event(pl, st) : 0; }

// Opt-in shared-memory sizes of every kernel that needs more than 48 KB, set once per DEVICE (cudaFuncSetAttribute acts
// on the current device's copy of the function; a per-process flag would leave a second device unset).  Called from the
// load / finalize / simulate entry points, never from a contract call.  *sm_count (may be null) receives the SM count.
int ensure_device_attrs(int *sm_count) {
    static std::mutex mu;
    static bool done[TQC_MAX_DEVICES] = {};
    static int sms[TQC_MAX_DEVICES] = {};
    int dev = 0;
    TQC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TQC_MAX_DEVICES) return fail(TQC_E_TOO_LARGE, "device ordinal beyond the library's table");
    std::lock_guard<std::mutex> lock(mu);
    if (!done[dev]) {
        TQC_CUDA(cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev));
        const auto dyn = cudaFuncAttributeMaxDynamicSharedMemorySize;
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tile_kernel<4, 4>, dyn, kMaxDynSmem));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tile_kernel<4, 1>, dyn, kMaxDynSmem));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tile_kernel<1, 4>, dyn, kMaxDynSmem));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tile_kernel<1, 1>, dyn, kMaxDynSmem));
        TQC_CUDA(cudaFuncSetAttribute(tqc::cross_mma_kernel<3>, dyn, 100 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::cross_mma_kernel<4>, dyn, 100 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::cross_mma_kernel<5>, dyn, 100 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::cross_mma_kernel<6>, dyn, 100 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tc_kernel<16>, dyn, 201 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tc_kernel<32>, dyn, 201 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tc_kernel<64>, dyn, 201 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tc_kernel<128>, dyn, 201 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::step_tc2_kernel<256>, dyn, 194 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::chain_kernel, dyn, 128 * 1024));
        TQC_CUDA(cudaFuncSetAttribute(tqc::sim_variant_kernel<false>, dyn, 24 << 13));
        TQC_CUDA(cudaFuncSetAttribute(tqc::sim_variant_kernel<false>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        done[dev] = true;
    }
    if (sm_count) *sm_count = sms[dev];
    return 0;
}

template <int MI, int MJ>
int launch_tile_t(const StepArgs &a, size_t smem, long long blocks, cudaStream_t st) {
    tqc::step_tile_kernel<MI, MJ><<<(unsigned)blocks, 256, smem, st>>>(a);
    TQC_CUDA(cudaGetLastError());
    return 0;
}

// Tile choice for the FFMA kernel: TI x TJ outputs per row, RPB rows per 256-thread block.
int launch_tile(tqc_plan_t *pl, StepArgs &a, int tag, cudaStream_t st) {
    const int MI = a.lgM >= 2 ? 4 : 1, MJ = a.lgN >= 2 ? 4 : 1;
    const long long M = 1ll << a.lgM, N = 1ll << a.lgN, K = 1ll << a.lgK;
    long long TI = MI == 4 ? std::min<long long>(M, 64) : M;
    long long capJ = 256ll * MJ * MI / TI;                 // threads per row-tile <= 256
    long long TJ = MJ == 4 ? std::min<long long>(std::min<long long>(N, capJ), 256) : N;
    if (MI == 4 && MJ == 4 && TJ < 64 && TI == 64 && M > 64) TI = std::min<long long>(M, std::min<long long>(256, 4096 / TJ));
    const long long tpr = (TI / MI) * (TJ / MJ);
    const long long RPB = std::max<long long>(1, 256 / tpr);
    long long TK = std::min<long long>(K, 16);
    const long long TIp = TI + (MI == 4 ? 4 : 1), TJp = TJ + (MJ == 4 ? 4 : 1);
    auto smem_of = [&](long long tk) { return (size_t)(8 * RPB * (TI + TJ) + 8 * (TI + TJ) + 4 * RPB * tk * (TIp + TJp) + 32); };
    while (TK > 1 && smem_of(TK) > (size_t)96 * 1024) TK /= 2;
    if (smem_of(TK) > (size_t)kMaxDynSmem) return fail(TQC_E_TOO_LARGE, "internal: tile does not fit shared memory");
    auto lg = [](long long v) { int l = 0; while ((1ll << l) < v) ++l; return l; };
    a.lgTI = lg(TI); a.lgTJ = lg(TJ); a.lgTK = lg(TK); a.lgRPB = lg(RPB);
    a.lgTilesI = lg(M / TI); a.lgTilesJ = lg(N / TJ);
    if ((1ll << a.lgTI) != TI || (1ll << a.lgTJ) != TJ || (1ll << a.lgTK) != TK || (1ll << a.lgRPB) != RPB)
        return fail(TQC_E_TOO_LARGE, "internal: tile dimensions must be powers of two");
    a.vec_store = (MJ == 4 && a.outB.n >= 1 && a.outB.src[0] == 0 && a.outB.dst[0] == 0 && a.outB.len[0] >= 2) ? 1 : 0;
    const long long rgroups = (a.R + RPB - 1) / RPB;
    const long long blocks = ((M / TI) * (N / TJ)) * rgroups;
    if (blocks <= 0 || blocks > 0x7fffffffll) return fail(TQC_E_TOO_LARGE, "step needs more than 2^31 thread blocks");
    int rc;
    if ((rc = note_launch(pl, tag, st))) return rc;
    if (MI == 4 && MJ == 4) rc = launch_tile_t<4, 4>(a, smem_of(TK), blocks, st);
    else if (MI == 4) rc = launch_tile_t<4, 1>(a, smem_of(TK), blocks, st);
    else if (MJ == 4) rc = launch_tile_t<1, 4>(a, smem_of(TK), blocks, st);
    else rc = launch_tile_t<1, 1>(a, smem_of(TK), blocks, st);
    return rc;
}

// outer digits of a node in its device order (most significant first): the layout minus the trailing inner digits
std::vector<int> outer_of(const Node &nd) { return std::vector<int>(nd.layout.begin(), nd.layout.end() - nd.n_inner); }

// digits of an operand's outer index (most significant first) -> bit positions inside C's row
void add_digit_scatter(BitPairs &bp, const std::vector<int> &outer, const std::vector<int> &c_layout) {
    const int no = (int)outer.size(), nc = (int)c_layout.size();
    for (int x = 0; x < no; ++x) {
        const int p = no - 1 - x;                                // digit position from the LSB side
        const int y = index_of(c_layout, outer[x]);
        const int pos = nc - 1 - y;
        bp.add_run(2 * p, 2 * pos, 2);
    }
}

// ---- cross mode (TABLE outputs; distribution mode and states-mode tables) --------------------
struct CrossCtx {
    int prefix_bits = 0;
    uint64_t prefix_value = 0;
    const std::vector<int> *free_bits = nullptr;      // per node (distribution) or null (all bits free)
    const std::vector<int64_t> *offsets = nullptr;    // per node float offsets (distribution)
    float *ws = nullptr;                               // base of table storage
    float *out = nullptr;                              // distribution root target
};

std::vector<int> free_qubits(const Node &v, int prefix_bits) {
    std::vector<int> f;
    for (int q : v.qubits) if (q >= prefix_bits) f.push_back(q);
    return f;
}

int build_cross_operand(tqc_plan_t *pl, const CrossCtx &cx, int v, const std::vector<int> &outer, OperandArgs &o,
                        int &lg_rows) {
    const HostPlan &hp = pl->hp;
    const Node &nd = hp.nodes[v];
    const std::vector<int> fq = free_qubits(nd, cx.prefix_bits);
    const int nd_bits = 2 * (int)outer.size();
    lg_rows = (int)fq.size() + nd_bits;
    o.keys = nullptr; o.in_or = 0; o.use_map = 0; o.in_map.n = 0;
    if (v < hp.m) {
        o.base = pl->d_leaf[v];
        if (fq.size() != nd.qubits.size()) {
            BitPairs bp;
            bp.add_run(0, 0, nd_bits);
            const int nq = (int)nd.qubits.size(), nf = (int)fq.size();
            unsigned long long fixed = 0;
            int t = 0;
            for (int pq = 0; pq < nq; ++pq) {
                const int q = nd.qubits[pq];
                const int keybit = nq - 1 - pq;
                if (q >= cx.prefix_bits) { bp.add(nd_bits + (nf - 1 - t), nd_bits + keybit); ++t; }
                else if ((cx.prefix_value >> (cx.prefix_bits - 1 - q)) & 1ull) fixed |= 1ull << (nd_bits + keybit);
            }
            if (!bp.build(o.in_map)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
            o.in_or = fixed;
            o.use_map = 1;
        }
    } else {
        const int64_t off = cx.offsets ? (*cx.offsets)[v] : nd.table_offset;
        o.base = cx.ws + off;
    }
    return 0;
}

int launch_cross_step(tqc_plan_t *pl, const CrossCtx &cx, int t, cudaStream_t st) {
    const HostPlan &hp = pl->hp;
    const Step &s = hp.steps[t];
    const int vc = hp.m + t;
    const Node &A = hp.nodes[s.lhs], &B = hp.nodes[s.rhs], &C = hp.nodes[vc];
    StepArgs a;
    memset(&a, 0, sizeof(a));
    int rc;
    if ((rc = build_cross_operand(pl, cx, s.lhs, s.outer_lhs, a.A, a.lgM))) return rc;
    if ((rc = build_cross_operand(pl, cx, s.rhs, s.outer_rhs, a.B, a.lgN))) return rc;
    a.lgK = 2 * (int)s.inner.size();
    a.R = 1;
    a.c_row_stride = 0;
    const std::vector<int> fa = free_qubits(A, cx.prefix_bits), fb = free_qubits(B, cx.prefix_bits);
    const bool dist_root = cx.out != nullptr && vc == hp.root();
    const int cdig = 2 * (int)C.layout.size();
    BitPairs pa, pb;
    add_digit_scatter(pa, outer_of(hp.nodes[s.lhs]), C.layout);
    add_digit_scatter(pb, outer_of(hp.nodes[s.rhs]), C.layout);
    const int na = 2 * (int)s.outer_lhs.size(), nb = 2 * (int)s.outer_rhs.size();
    if (dist_root) {
        // product-order row bits -> global bit order: free qubits ascending, lowest id = MSB (G4)
        std::vector<int> all = fa;
        all.insert(all.end(), fb.begin(), fb.end());
        auto dst_of = [&](int q) { int c = 0; for (int x : all) if (x > q) ++c; return c; };
        for (size_t i = 0; i < fa.size(); ++i) pa.add(na + (int)(fa.size() - 1 - i), dst_of(fa[i]));
        for (size_t i = 0; i < fb.size(); ++i) pb.add(nb + (int)(fb.size() - 1 - i), dst_of(fb[i]));
        a.C = cx.out;
    } else {
        pa.add_run(na, cdig + (int)fb.size(), (int)fa.size());
        pb.add_run(nb, cdig, (int)fb.size());
        const int64_t off = cx.offsets ? (*cx.offsets)[vc] : C.table_offset;
        a.C = cx.ws + off;
    }
    if (!pa.build(a.outA) || !pb.build(a.outB)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
    // short bond, many rows on both sides: warp-level 3xTF32 tensor-core tiles (kernels_cross.cuh)
    if (pl->use_tcgen05 >= 0 && a.lgK >= 3 && a.lgK <= 6 && std::min(a.lgM, a.lgN) >= 6 && std::max(a.lgM, a.lgN) >= 7 &&
        !dev_env("TQC_NO_CROSS_MMA")) {
        if (a.lgN < 7) { std::swap(a.A, a.B); std::swap(a.outA, a.outB); std::swap(a.lgM, a.lgN); }
        a.lgTilesI = a.lgM - 6; a.lgTilesJ = a.lgN - 7;
        a.vec_store = (a.outB.n >= 1 && a.outB.src[0] == 0 && a.outB.dst[0] == 0 && a.outB.len[0] >= 2) ? 1 : 0;
        if (a.vec_store && !dev_env("TQC_CROSS_STAGED")) a.vec_store = 2;          // 8-byte stores straight from the fragments
        const long long blocks = 1ll << (a.lgTilesI + a.lgTilesJ);
        if (blocks > 0x7fffffffll) return fail(TQC_E_TOO_LARGE, "step needs more than 2^31 thread blocks");
        const size_t smem = tqc::cross_mma_smem(a.lgK, a.vec_store != 2);
        if ((rc = note_launch(pl, t, st))) return rc;
        switch (a.lgK) {
            case 3: tqc::cross_mma_kernel<3><<<(unsigned)blocks, 256, smem, st>>>(a); break;
            case 4: tqc::cross_mma_kernel<4><<<(unsigned)blocks, 256, smem, st>>>(a); break;
            case 5: tqc::cross_mma_kernel<5><<<(unsigned)blocks, 256, smem, st>>>(a); break;
            default: tqc::cross_mma_kernel<6><<<(unsigned)blocks, 256, smem, st>>>(a); break;
        }
        TQC_CUDA(cudaGetLastError());
        return 0;
    }
    return launch_tile(pl, a, t, st);
}

// ---- batch mode (one row per state of the chunk) ---------------------------------------------
struct BatchCtx {
    float *tables = nullptr;     // states-mode table region
    uint32_t *keys = nullptr;    // [n_slots][cap]
    float *batch = nullptr;      // BATCH intermediates: node block at ws_offset * cap
    long long cap = 0;
    int R = 0;
    float *out = nullptr;        // out + chunk_start
};

void batch_operand(tqc_plan_t *pl, const BatchCtx &bx, int v, const float *&base, const uint32_t *&keys) {
    const HostPlan &hp = pl->hp;
    const Node &nd = hp.nodes[v];
    if (nd.kind == tqc::NODE_BATCH) { base = bx.batch + nd.ws_offset * bx.cap; keys = nullptr; }
    else {
        base = v < hp.m ? pl->d_leaf[v] : bx.tables + nd.table_offset;
        keys = bx.keys + (long long)nd.key_slot * bx.cap;
    }
}

// ---- tensor-pipe step (kernels_tc.cuh) ----------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode_fn(EncodeTiledFn *out) {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        TQC_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres));
        if (!p || qres != cudaDriverEntryPointSuccess) return fail(TQC_E_CUDA, "cuTensorMapEncodeTiled not available in this driver");
        fn = (EncodeTiledFn)p;
    }
    *out = fn;
    return 0;
}

// operand seen as a 3-D fp32 tensor {K, rows_inner, rows_outer}: one {32, box_rows, 1} box per TMA load
int make_operand_map(CUtensorMap *map, const float *base, int lgK, int lgRows, long long n_outer, int box_rows) {
    EncodeTiledFn enc;
    int rc = get_encode_fn(&enc);
    if (rc) return rc;
    const cuuint64_t dims[3] = {(cuuint64_t)1 << lgK, (cuuint64_t)1 << lgRows, (cuuint64_t)std::max<long long>(n_outer, 1)};
    const cuuint64_t strides[2] = {((cuuint64_t)4) << lgK, ((cuuint64_t)4) << (lgK + lgRows)};
    const cuuint32_t box[3] = {(cuuint32_t)tqc::TC_BK, (cuuint32_t)box_rows, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)base, dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(TQC_E_CUDA, "cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
    return 0;
}

bool tc_eligible(int lgM, int lgN, int lgK) {
    if (std::max(lgM, lgN) > 14) return false;                  // at most 256 tiles per side (C-offset tables of the kernel)
    if (lgK == 4 && lgM >= 8 && lgN >= 8) return dev_env("TQC_TC_NO_PAIR") == nullptr && dev_env("TQC_TC_NO_K16") == nullptr;   // K = 16 on the CTA-pair kernel (half of each k-block is zero fill)
    return lgK >= 5 && std::max(lgM, lgN) >= 7 && std::min(lgM, lgN) >= 4;
}

struct TcOperand { const float *base; const uint32_t *keys; long long n_outer; };

int launch_tc_step(tqc_plan_t *pl, TcOperand A, TcOperand B, BitMap outA, BitMap outB, int lgM, int lgN, int lgK, float *C,
                   long long c_row_stride, int R, int tag, cudaStream_t st) {
    const int sm_count = pl->sm_count > 0 ? pl->sm_count : 148;
    auto has_bit0 = [](const BitMap &m) { for (int s = 0; s < m.n; ++s) if (m.dst[s] == 0) return true; return false; };
    // CTA-pair kernel (kernels_tc2.cuh): 256 x BN tiles over two SMs.  The M side needs >= 256 rows, the N side >= 128; with
    // both orientations possible the N side is the operand that owns C's lowest offset bit (8- or 16-byte stores from registers).
    static const bool no_pair = dev_env("TQC_TC_NO_PAIR") != nullptr;
    {
        // (64-column pair tiles were tried: a k-block then holds 384 cycles of MMAs against about 1800 cycles of fixed pipeline
        // hand-shake per k-block, no gain over step_tc_kernel<64>; those steps are bound by streaming their 16 MB operand)
        const bool keep_ok = lgM >= 8 && lgN >= 8, swap_ok = keep_ok;          // outer dimensions are powers of four
        if (!no_pair && lgK >= 4 && (keep_ok || swap_ok)) {
            bool sw = !keep_ok;
            if (keep_ok && swap_ok) sw = has_bit0(outA);
            if (sw) { std::swap(A, B); std::swap(outA, outB); std::swap(lgM, lgN); }
            tqc::TcArgs a;
            memset(&a, 0, sizeof(a));
            a.keysA = A.keys; a.keysB = B.keys;
            a.C = C; a.c_row_stride = c_row_stride;
            a.outA = outA; a.outB = outB;
            a.lgM = lgM; a.lgN = lgN; a.lgK = lgK; a.R = R;
            a.BN = 256;
            { const char *dbg = dev_env("TQC_TC_DEBUG"); a.debug = dbg ? std::atoi(dbg) : 0; }
            a.mask_hi = 1;
            if (const char *tp = dev_env("TQC_TC_TRACE_PTR")) a.trace = (unsigned long long *)std::strtoull(tp, nullptr, 0);
            // columns j, j + 1 adjacent in C: 1; j .. j + 3 (j a multiple of 4): 2 (16-byte stores after a lane exchange)
            a.vec4 = (outB.n >= 1 && outB.src[0] == 0 && outB.dst[0] == 0) ? (outB.len[0] >= 2 ? 2 : 1) : 0;
            const size_t stage_bytes = 2 * (size_t)128 * tqc::TC_BK * 4 + 2 * (size_t)(a.BN / 2) * tqc::TC_BK * 4;
            a.stages = (int)std::min<size_t>(6, (192 * 1024) / stage_bytes);
            if (const char *sv = dev_env("TQC_TC_STAGES")) a.stages = std::max(2, std::min(a.stages, std::atoi(sv)));
            CUtensorMap mapA, mapB;
            int rc;
            if ((rc = make_operand_map(&mapA, A.base, lgK, lgM, A.n_outer, 128))) return rc;
            if ((rc = make_operand_map(&mapB, B.base, lgK, lgN, B.n_outer, a.BN / 2))) return rc;
            const long long total = (1ll << (lgM - 8)) * ((1ll << lgN) / a.BN) * (long long)R;
            const unsigned grid = 2u * (unsigned)std::min<long long>(total, sm_count / 2);
            if (dev_env("TQC_TC_TRACE"))
            {
                fprintf(stderr, "tc2 step %d: lgM %d lgN %d lgK %d swap %d BN %d vec2 %d R %d stages %d  outA", tag, lgM, lgN, lgK, (int)sw, a.BN, a.vec4, R, a.stages);
                for (int q = 0; q < outA.n; ++q) fprintf(stderr, " %d+%d>%d", outA.src[q], outA.len[q], outA.dst[q]);
                fprintf(stderr, "  outB");
                for (int q = 0; q < outB.n; ++q) fprintf(stderr, " %d+%d>%d", outB.src[q], outB.len[q], outB.dst[q]);
                fprintf(stderr, "\n");
            }
            if ((rc = note_launch(pl, tag, st))) return rc;
            const size_t smem = a.stages * stage_bytes + 1024;
            pl->pair_launches++;
            tqc::step_tc2_kernel<256><<<grid, tqc::tc2_threads(256), smem, st>>>(mapA, mapB, a);
            TQC_CUDA(cudaGetLastError());
            return 0;
        }
    }
    if (lgK < 5) return fail(TQC_E_TOO_LARGE, "internal: a K = 16 tensor-pipe step needs the CTA-pair kernel");
    // the M side needs >= 128 rows; with both sides large, the N side (vector stores run along it) takes C's lowest bits
    bool swap = lgM < 7;
    if (lgM >= 7 && lgN >= 7 && has_bit0(outA)) swap = true;
    if (swap) { std::swap(A, B); std::swap(outA, outB); std::swap(lgM, lgN); }
    tqc::TcArgs a;
    memset(&a, 0, sizeof(a));
    a.keysA = A.keys; a.keysB = B.keys;
    a.C = C; a.c_row_stride = c_row_stride;
    a.outA = outA; a.outB = outB;
    a.lgM = lgM; a.lgN = lgN; a.lgK = lgK; a.R = R;
    a.BN = (int)std::min<long long>(128, 1ll << lgN);
    { const char *dbg = dev_env("TQC_TC_DEBUG"); a.debug = dbg ? std::atoi(dbg) : 0; }
    { const char *ck = dev_env("TQC_TC_CHUNK"); a.chunk_kb = ck ? std::atoi(ck) : 0; }
    // hi parts rounded to nearest (rewritten in shared memory): removes the systematic -2.4e-7 per step of the truncating
    // split (dropped lo*lo and truncated lo are then zero-mean).  TQC_TC_TRUNC=1 keeps the raw tile as hi (measurements).
    a.mask_hi = dev_env("TQC_TC_TRUNC") ? 0 : 1;
    const size_t stage_bytes = 2 * (size_t)tqc::TC_BM * tqc::TC_BK * 4 + 2 * (size_t)a.BN * tqc::TC_BK * 4;
    a.stages = (int)std::min<size_t>(4, (200 * 1024) / stage_bytes);     // + 24 KB static (epilogue scratch, tables)
    a.vec4 = (outB.n >= 1 && outB.src[0] == 0 && outB.dst[0] == 0 && outB.len[0] >= 2) ? 1 : 0;
    CUtensorMap mapA, mapB;
    int rc;
    if ((rc = make_operand_map(&mapA, A.base, lgK, lgM, A.n_outer, tqc::TC_BM))) return rc;
    if ((rc = make_operand_map(&mapB, B.base, lgK, lgN, B.n_outer, a.BN))) return rc;
    const long long total = (1ll << (lgM - 7)) * ((1ll << lgN) / a.BN) * (long long)R;
    const unsigned grid = (unsigned)std::min<long long>(total, sm_count);
    if (dev_env("TQC_TC_TRACE"))
        fprintf(stderr, "tc step %d: lgM %d lgN %d lgK %d swap %d vec4 %d keyedA %d keyedB %d R %d outB.n %d outB[0]=(%d,%d,%d)\n", tag, lgM, lgN, lgK,
                (int)swap, a.vec4, A.keys != nullptr, B.keys != nullptr, R, outB.n, outB.src[0], outB.dst[0], outB.len[0]);
    if ((rc = note_launch(pl, tag, st))) return rc;
    const size_t smem = a.stages * stage_bytes + 1024;
    switch (a.BN) {
        case 16: tqc::step_tc_kernel<16><<<grid, tqc::TC_THREADS, smem, st>>>(mapA, mapB, a); break;
        case 32: tqc::step_tc_kernel<32><<<grid, tqc::TC_THREADS, smem, st>>>(mapA, mapB, a); break;
        case 64: tqc::step_tc_kernel<64><<<grid, tqc::TC_THREADS, smem, st>>>(mapA, mapB, a); break;
        default: tqc::step_tc_kernel<128><<<grid, tqc::TC_THREADS, smem, st>>>(mapA, mapB, a); break;
    }
    TQC_CUDA(cudaGetLastError());
    return 0;
}

int launch_batch_step(tqc_plan_t *pl, const BatchCtx &bx, int t, cudaStream_t st) {
    const HostPlan &hp = pl->hp;
    const Step &s = hp.steps[t];
    const int vc = hp.m + t;
    const Node &C = hp.nodes[vc];
    const int lgM = 2 * (int)s.outer_lhs.size(), lgN = 2 * (int)s.outer_rhs.size(), lgK = 2 * (int)s.inner.size();
    float *cbase = (vc == hp.root()) ? bx.out : bx.batch + C.ws_offset * bx.cap;
    if (lgM == 0 && lgN == 0) {
        DotArgs d;
        memset(&d, 0, sizeof(d));
        batch_operand(pl, bx, s.lhs, d.A, d.keysA);
        batch_operand(pl, bx, s.rhs, d.B, d.keysB);
        d.out = cbase; d.lgK = lgK; d.R = bx.R;
        long long G = std::min<long long>(32, std::max<long long>(1, (1ll << lgK) / 4));
        const long long rows_per_block = (32 / G) * 8;
        const long long blocks = (bx.R + rows_per_block - 1) / rows_per_block;
        int rc = note_launch(pl, t, st);
        if (rc) return rc;
        tqc::dot_kernel<<<(unsigned)blocks, 256, 0, st>>>(d);
        TQC_CUDA(cudaGetLastError());
        return 0;
    }
    StepArgs a;
    memset(&a, 0, sizeof(a));
    batch_operand(pl, bx, s.lhs, a.A.base, a.A.keys);
    batch_operand(pl, bx, s.rhs, a.B.base, a.B.keys);
    a.lgM = lgM; a.lgN = lgN; a.lgK = lgK;
    a.R = bx.R;
    a.C = cbase;
    a.c_row_stride = 1ll << (2 * (int)C.open.size());
    BitPairs pa, pb;
    add_digit_scatter(pa, outer_of(hp.nodes[s.lhs]), C.layout);
    add_digit_scatter(pb, outer_of(hp.nodes[s.rhs]), C.layout);
    if (!pa.build(a.outA) || !pb.build(a.outB)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
    if (s.kernel_class == TQC_KERNEL_TCGEN05) {
        auto n_outer = [&](int v) -> long long {
            const Node &nd = hp.nodes[v];
            return nd.kind == tqc::NODE_BATCH ? (long long)bx.R : (1ll << (int)nd.qubits.size());
        };
        TcOperand oa{a.A.base, a.A.keys, n_outer(s.lhs)}, ob{a.B.base, a.B.keys, n_outer(s.rhs)};
        return launch_tc_step(pl, oa, ob, a.outA, a.outB, lgM, lgN, lgK, cbase, a.c_row_stride, bx.R, t, st);
    }
    return launch_tile(pl, a, t, st);
}

// ---- fused chain: plan-time step table --------------------------------------------------------
// Eligible when every per-state (BATCH) step has at most 1024 outputs and small operands, so that all intermediates
// of one state fit a warp's shared-memory scratch.
bool build_chain(tqc_plan_t *pl) {
    const HostPlan &hp = pl->hp;
    if (hp.mode != TQC_MODE_STATES || hp.m < 2 || hp.nodes[hp.root()].kind != tqc::NODE_BATCH) return false;
    if (hp.n_key_slots > 32) return false;
    std::vector<int> bsteps;
    for (int t = 0; t < hp.m - 1; ++t) if (hp.nodes[hp.m + t].kind == tqc::NODE_BATCH) bsteps.push_back(t);
    if (bsteps.empty() || (int)bsteps.size() > tqc::CHAIN_MAX_STEPS) return false;
    auto pad = [](long long floats, int lgK) { return lgK >= 2 ? floats + ((floats >> lgK) << 2) : floats; };
    auto align4 = [](long long v) { return (v + 3) / 4 * 4; };
    std::vector<tqc::ChainStep> tab;
    std::vector<int> leafA, leafB, g_leaf;
    std::vector<tqc::ChainGather> gathers;
    std::vector<long long> node_ofs(hp.nodes.size(), -1);
    long long top = 0, stop = 0, f4 = 0, tab_entries = 0;      // intermediates / staged operands / float4s / table entries
    for (int t : bsteps) {
        const Step &s = hp.steps[t];
        const int vc = hp.m + t;
        const Node &C = hp.nodes[vc];
        const int lgM = 2 * (int)s.outer_lhs.size(), lgN = 2 * (int)s.outer_rhs.size(), lgK = 2 * (int)s.inner.size();
        if (lgM + lgN > 10) return false;
        tqc::ChainStep cs;
        memset(&cs, 0, sizeof(cs));
        cs.lgM = lgM; cs.lgN = lgN; cs.lgK = lgK;
        int la = -1, lb = -1;
        for (int side = 0; side < 2; ++side) {
            const int v = side ? s.rhs : s.lhs;
            const Node &nd = hp.nodes[v];
            tqc::ChainOperand &o = side ? cs.B : cs.A;
            const int lgRows = side ? lgN : lgM, lgOther = side ? lgM : lgN;
            const long long floats = 1ll << (lgRows + lgK);
            o.table_ofs = -1;
            if (nd.kind == tqc::NODE_BATCH) {
                if (node_ofs[v] < 0) return false;
                o.gathered = 0;
                o.smem_ofs = (int)node_ofs[v];
                o.pitch = (1 << lgK) + (lgK >= 2 ? 4 : 0);
            } else {
                o.gathered = 1;
                o.key_slot = nd.key_slot;
                if (v < hp.m) (side ? lb : la) = v; else o.table_ofs = nd.table_offset;
                const bool reuse = lgOther > 0;
                o.staged = (reuse && floats >= 4 && floats <= 1024) ? 1 : 0;
                if (!o.staged && reuse && floats > 16384) return false;
                o.pitch = (1 << lgK) + ((o.staged && lgK >= 2) ? 4 : 0);
                if (o.staged) {
                    if ((int)gathers.size() >= tqc::CHAIN_MAX_GATHER) return false;
                    tqc::ChainGather gg;
                    memset(&gg, 0, sizeof(gg));
                    gg.table_ofs = o.table_ofs; gg.key_slot = nd.key_slot; gg.lg_floats = lgRows + lgK; gg.lgK = lgK;
                    gg.smem_ofs = (int)stop; gg.f4_begin = (int)f4;
                    o.smem_ofs = (int)stop;
                    stop += align4(pad(floats, lgK));
                    f4 += floats / 4;
                    gathers.push_back(gg);
                    g_leaf.push_back(v < hp.m ? v : -1);
                }
            }
        }
        if (vc == hp.root()) { cs.c_smem_ofs = -1; cs.c_lgK = 0; }
        else {
            const int c_lgK = 2 * (int)hp.steps[C.consumer].inner.size();
            const long long floats = 1ll << (2 * (int)C.open.size());
            if (floats > 4096) return false;
            cs.c_smem_ofs = (int)top; cs.c_lgK = c_lgK;
            node_ofs[vc] = top;
            top += align4(pad(floats, c_lgK));
        }
        cs.tab_ofs = (int)tab_entries;
        tab_entries += (1ll << lgM) + (1ll << lgN);
        BitPairs pa, pb;
        add_digit_scatter(pa, outer_of(hp.nodes[s.lhs]), C.layout);
        add_digit_scatter(pb, outer_of(hp.nodes[s.rhs]), C.layout);
        if (!pa.build(cs.outA) || !pb.build(cs.outB)) return false;
        tab.push_back(cs); leafA.push_back(la); leafB.push_back(lb);
    }
    if (top + 2 * stop > 3072 || f4 > 32ll * tqc::CHAIN_MAX_F4 || tab_entries > 8192) return false;   // 12 KB of scratch per warp
    pl->chain_host = tab; pl->chain_leafA = leafA; pl->chain_leafB = leafB;
    pl->chain_gather = gathers; pl->chain_gather_leaf = g_leaf;
    pl->chain_scratch = (int)(top + 2 * stop); pl->chain_stage = (int)stop; pl->chain_f4 = (int)f4; pl->chain_tab_entries = (int)tab_entries;
    return true;
}

// ---- plan-specialised chain kernel: source generation + NVRTC + driver module ---------------------
// The generated translation unit includes kernels_chain.cuh and defines ChainPlanSpec::run as the plan's steps in
// straight-line form (chain_step_spec<...> per step, every shape, pitch, offset and index map a literal).
struct JitApi {
    void *nvrtc = nullptr;
    nvrtcResult (*CreateProgram)(nvrtcProgram *, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
    nvrtcResult (*CompileProgram)(nvrtcProgram, int, const char *const *) = nullptr;
    nvrtcResult (*GetProgramLogSize)(nvrtcProgram, size_t *) = nullptr;
    nvrtcResult (*GetProgramLog)(nvrtcProgram, char *) = nullptr;
    nvrtcResult (*GetCUBINSize)(nvrtcProgram, size_t *) = nullptr;
    nvrtcResult (*GetCUBIN)(nvrtcProgram, char *) = nullptr;
    nvrtcResult (*DestroyProgram)(nvrtcProgram *) = nullptr;
    CUresult (*ModuleLoadData)(CUmodule *, const void *) = nullptr;
    CUresult (*ModuleGetFunction)(CUfunction *, CUmodule, const char *) = nullptr;
    CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
    CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream, void **, void **) = nullptr;
    CUresult (*ModuleUnload)(CUmodule) = nullptr;
    bool ok = false;
    std::string why;
};

JitApi &jit_api() {
    static JitApi api;
    static bool tried = false;
    if (tried) return api;
    tried = true;
    const char *names[] = {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"};
    for (const char *n : names) if ((api.nvrtc = dlopen(n, RTLD_NOW | RTLD_LOCAL))) break;
    if (!api.nvrtc) { api.why = "libnvrtc not found"; return api; }
#define TQC_SYM(field, sym) *(void **)(&api.field) = dlsym(api.nvrtc, sym); if (!api.field) { api.why = std::string("missing ") + sym; return api; }
    TQC_SYM(CreateProgram, "nvrtcCreateProgram") TQC_SYM(CompileProgram, "nvrtcCompileProgram")
    TQC_SYM(GetProgramLogSize, "nvrtcGetProgramLogSize") TQC_SYM(GetProgramLog, "nvrtcGetProgramLog")
    TQC_SYM(GetCUBINSize, "nvrtcGetCUBINSize") TQC_SYM(GetCUBIN, "nvrtcGetCUBIN") TQC_SYM(DestroyProgram, "nvrtcDestroyProgram")
#undef TQC_SYM
    auto drv = [&](const char *sym, void **out) {
        cudaDriverEntryPointQueryResult q;
        return cudaGetDriverEntryPoint(sym, out, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess && *out;
    };
    if (!drv("cuModuleLoadData", (void **)&api.ModuleLoadData) || !drv("cuModuleGetFunction", (void **)&api.ModuleGetFunction) ||
        !drv("cuFuncSetAttribute", (void **)&api.FuncSetAttribute) || !drv("cuLaunchKernel", (void **)&api.LaunchKernel) ||
        !drv("cuModuleUnload", (void **)&api.ModuleUnload)) { api.why = "driver entry points not available"; return api; }
    api.ok = true;
    return api;
}

std::string bitmap_expr(const BitMap &m, const char *var) {
    if (m.n == 0) return "0";
    std::string e;
    for (int s = 0; s < m.n; ++s) {
        if (s) e += " | ";
        e += "(((" + std::string(var) + " >> " + std::to_string((int)m.src[s]) + ") & " + std::to_string((1 << m.len[s]) - 1) + ") << " +
             std::to_string((int)m.dst[s]) + ")";
    }
    return e;
}

std::string chain_source(const tqc_plan_t *pl) {
    std::string src = "#include \"kernels_chain.cuh\"\nnamespace tqc {\nstruct ChainPlanSpec {\n"
                      "  static __device__ __forceinline__ void run(const ChainStateCtx &c) {\n";
    for (size_t t = 0; t < pl->chain_host.size(); ++t) {
        const tqc::ChainStep &s = pl->chain_host[t];
        auto operand = [&](const tqc::ChainOperand &o, const char *which, int lgRows) {
            if (!o.gathered) return "c.inter + " + std::to_string(o.smem_ofs);
            if (o.staged) return "c.stg + " + std::to_string(o.smem_ofs);
            const std::string base = o.table_ofs >= 0 ? "c.a->tables + " + std::to_string(o.table_ofs) + "ll"
                                                      : "c.steps[" + std::to_string(t) + "]." + which + ".base";
            return "(" + base + ") + ((size_t)__shfl_sync(0xffffffffu, c.mykey, " + std::to_string(o.key_slot) + ") << " +
                   std::to_string(lgRows + s.lgK) + ")";
        };
        // a bond-wide operand read straight from global memory with a single row on the other side: row-split step
        // (coalesced reads); if that operand is A, the roles are swapped in the generated call
        const bool direct_a = s.A.gathered && !s.A.staged, direct_b = s.B.gathered && !s.B.staged;
        const bool split_b = direct_b && s.lgM == 0 && s.lgK >= 4 && s.lgN >= 1;
        const bool split_a = !split_b && direct_a && s.lgN == 0 && s.lgK >= 4 && s.lgM >= 1;
        if (split_a) {
            src += "    { const float *pa = " + operand(s.B, "B", s.lgN) + ";\n      const float *pb = " + operand(s.A, "A", s.lgM) + ";\n";
            src += "      chain_step_spec<0, " + std::to_string(s.lgM) + ", " + std::to_string(s.lgK) + ", " + std::to_string(s.B.pitch) + ", " +
                   std::to_string(s.A.pitch) + ", true>(pa, pb, c.lane, [&](int j, int i, float v) {\n";
        } else {
            src += "    { const float *pa = " + operand(s.A, "A", s.lgM) + ";\n      const float *pb = " + operand(s.B, "B", s.lgN) + ";\n";
            src += "      chain_step_spec<" + std::to_string(s.lgM) + ", " + std::to_string(s.lgN) + ", " + std::to_string(s.lgK) + ", " +
                   std::to_string(s.A.pitch) + ", " + std::to_string(s.B.pitch) + (split_b ? ", true" : "") + ">(pa, pb, c.lane, [&](int i, int j, float v) {\n";
        }
        if (s.c_smem_ofs < 0) src += "        *c.out_r = v;\n";
        else {
            src += "        const int x = (" + bitmap_expr(s.outA, "i") + ") | (" + bitmap_expr(s.outB, "j") + ");\n";
            src += "        c.inter[" + std::to_string(s.c_smem_ofs) + " + " +
                   (s.c_lgK >= 2 ? "x + ((x >> " + std::to_string(s.c_lgK) + ") << 2)" : std::string("x")) + "] = v;\n";
        }
        src += "      });\n      __syncwarp(); }\n";
    }
    src += "  }\n";
    // the staged operands of one state: for every 32-chunk slot the lane ranges of the gathers it covers, with the row
    // size, the padding and the destination as constants (the generic kernel reads the same from a shared-memory table)
    if (dev_env("TQC_CHAIN_TABLE_GATHER")) src += "  static constexpr bool kOwnGather = false;\n  static __device__ __forceinline__ void gather(const ChainArgs &, uint32_t, uint32_t, int) {}\n";
    else {
        src += "  static constexpr bool kOwnGather = true;\n"
               "  static __device__ __forceinline__ void gather(const ChainArgs &a, uint32_t key, uint32_t dst, int lane) {\n";
        const int ng = (int)pl->chain_gather.size();
        for (int gi = 0; gi < ng; ++gi) {
            const tqc::ChainGather &gg = pl->chain_gather[gi];
            const std::string base = gg.table_ofs >= 0 ? "a.tables + " + std::to_string(gg.table_ofs) + "ll" : "a.g[" + std::to_string(gi) + "].base";
            src += "    const float *s" + std::to_string(gi) + " = (" + base + ") + ((size_t)__shfl_sync(0xffffffffu, key, " +
                   std::to_string(gg.key_slot) + ") << " + std::to_string(gg.lg_floats) + ");\n";
        }
        for (int q = 0; q * 32 < pl->chain_f4; ++q) {
            for (int gi = 0; gi < ng; ++gi) {
                const tqc::ChainGather &gg = pl->chain_gather[gi];
                const int f_end = gi + 1 < ng ? pl->chain_gather[gi + 1].f4_begin : pl->chain_f4;
                const int lo = std::max(gg.f4_begin, q * 32), hi = std::min(f_end, q * 32 + 32);
                if (lo >= hi) continue;
                const int l0 = lo - q * 32, l1 = hi - q * 32, c0 = lo - gg.f4_begin;
                const std::string cexp = std::to_string(c0 - l0) + " + lane";
                const std::string pad = gg.lgK >= 2 ? "x + ((x >> " + std::to_string(gg.lgK) + ") << 2)" : std::string("x");
                src += "    " + (l0 == 0 && l1 == 32 ? std::string("") : "if (lane >= " + std::to_string(l0) + " && lane < " + std::to_string(l1) + ") ") +
                       "{ const int x = 4 * (" + cexp + "); chain_cp16(dst + 4u * (uint32_t)(" + std::to_string(gg.smem_ofs) + " + " + pad +
                       "), s" + std::to_string(gi) + " + x); }\n";
            }
        }
        src += "  }\n";
    }
    src += "};\n}  // namespace tqc\n"
           "extern \"C\" __global__ void __launch_bounds__(256, 3) chain_spec_kernel(const tqc::ChainArgs a) {\n"
           "  tqc::chain_body<tqc::ChainPlanSpec>(a);\n}\n";
    return src;
}

// fills pl->jit_fn, or leaves it null with the reason in pl->jit_note (the interpreter kernel then runs the chain)
void chain_jit_build(tqc_plan_t *pl) {
    JitApi &api = jit_api();
    if (!api.ok) { pl->jit_note = "chain kernel not specialised: " + api.why; return; }
    Dl_info info;
    if (!dladdr((void *)&tqc_version, &info) || !info.dli_fname) { pl->jit_note = "chain kernel not specialised: library path unknown"; return; }
    std::string dir(info.dli_fname);
    dir = dir.substr(0, dir.find_last_of('/')) + "/csrc";
    const std::string src = chain_source(pl);
    nvrtcProgram prog;
    if (api.CreateProgram(&prog, src.c_str(), "chain_spec.cu", 0, nullptr, nullptr) != NVRTC_SUCCESS) { pl->jit_note = "nvrtcCreateProgram failed"; return; }
    const std::string inc = "-I" + dir;
    const char *opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", inc.c_str(), "-lineinfo", "-DTQC_CHAIN_NO_MMA"};
    if (dev_env("TQC_MMA_MASK_LO")) opts[4] = "-DTQC_MMA_MASK_LO";
    const nvrtcResult rc = api.CompileProgram(prog, dev_env("TQC_CHAIN_NO_MMA") || dev_env("TQC_MMA_MASK_LO") ? 5 : 4, opts);
    if (rc != NVRTC_SUCCESS) {
        size_t n = 0;
        api.GetProgramLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) api.GetProgramLog(prog, &log[0]);
        pl->jit_note = "chain kernel not specialised: compile failed: " + log.substr(0, 2000);
        api.DestroyProgram(&prog);
        return;
    }
    size_t n = 0;
    api.GetCUBINSize(prog, &n);
    std::vector<char> cubin(n);
    api.GetCUBIN(prog, cubin.data());
    api.DestroyProgram(&prog);
    CUmodule mod;
    CUfunction fn;
    if (api.ModuleLoadData(&mod, cubin.data()) != CUDA_SUCCESS) { pl->jit_note = "chain kernel not specialised: cuModuleLoadData failed"; return; }
    if (api.ModuleGetFunction(&fn, mod, "chain_spec_kernel") != CUDA_SUCCESS ||
        api.FuncSetAttribute(fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, 128 * 1024) != CUDA_SUCCESS) {
        api.ModuleUnload(mod);
        pl->jit_note = "chain kernel not specialised: kernel not found in module";
        return;
    }
    pl->jit_module = (void *)mod; pl->jit_fn = (void *)fn;
    pl->jit_note = "chain kernel specialised for this plan (" + std::to_string(src.size()) + " bytes of generated source)";
}

int ensure_chain(tqc_plan_t *pl) {
    if (!pl->chain || pl->d_chain) return 0;
    std::vector<tqc::ChainStep> tab = pl->chain_host;
    for (size_t x = 0; x < tab.size(); ++x) {
        if (pl->chain_leafA[x] >= 0) tab[x].A.base = pl->d_leaf[pl->chain_leafA[x]];
        if (pl->chain_leafB[x] >= 0) tab[x].B.base = pl->d_leaf[pl->chain_leafB[x]];
    }
    TQC_CUDA(cudaMalloc(&pl->d_chain, tab.size() * sizeof(tqc::ChainStep)));
    TQC_CUDA(cudaMemcpy(pl->d_chain, tab.data(), tab.size() * sizeof(tqc::ChainStep), cudaMemcpyHostToDevice));
    if (pl->chain_mode == 0) chain_jit_build(pl);
    return 0;
}

int ensure_meta(tqc_plan_t *pl) {
    if (pl->d_slot_ofs || pl->hp.mode != TQC_MODE_STATES || pl->hp.n_key_slots == 0) return 0;
    const HostPlan &hp = pl->hp;
    std::vector<int32_t> ofs(hp.n_key_slots + 1, 0), qs;
    for (int slot = 0; slot < hp.n_key_slots; ++slot) {
        for (const Node &nd : hp.nodes)
            if (nd.key_slot == slot) for (int q : nd.qubits) qs.push_back(q);
        ofs[slot + 1] = (int32_t)qs.size();
    }
    TQC_CUDA(cudaMalloc(&pl->d_slot_ofs, ofs.size() * sizeof(int32_t)));
    TQC_CUDA(cudaMalloc(&pl->d_slot_qubits, std::max<size_t>(1, qs.size()) * sizeof(int32_t)));
    TQC_CUDA(cudaMemcpy(pl->d_slot_ofs, ofs.data(), ofs.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    if (!qs.empty()) TQC_CUDA(cudaMemcpy(pl->d_slot_qubits, qs.data(), qs.size() * sizeof(int32_t), cudaMemcpyHostToDevice));
    return 0;
}

size_t align256(size_t v) { return (v + 255) / 256 * 256; }
// decides once whether the table steps of a states-mode plan fork onto side streams, and creates the streams / events
int ensure_lanes(tqc_plan_t *pl) {
    if (pl->tables_parallel >= 0) return 0;
    const HostPlan &hp = pl->hp;
    int n_tab = 0;
    bool leaf_only = true;
    for (int t = 0; t < hp.m - 1; ++t) {
        if (hp.nodes[hp.m + t].kind != tqc::NODE_TABLE) continue;
        ++n_tab;
        if (hp.steps[t].lhs >= hp.m || hp.steps[t].rhs >= hp.m) leaf_only = false;
    }
    pl->tables_parallel = (hp.mode == TQC_MODE_STATES && n_tab >= 1 && leaf_only && !dev_env("TQC_NO_FORK")) ? 1 : 0;
    if (pl->tables_parallel) {
        TQC_CUDA(cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming));
        for (int l = 0; l < tqc_plan::N_LANES; ++l) {
            TQC_CUDA(cudaStreamCreateWithFlags(&pl->lane[l], cudaStreamNonBlocking));
            TQC_CUDA(cudaEventCreateWithFlags(&pl->ev_join[l], cudaEventDisableTiming));
        }
    }
    return 0;
}


// states-mode workspace: [tables][keys: n_slots x cap u32][batch: ws_floats_per_state x cap]
size_t states_fixed_bytes(const HostPlan &hp) { return align256((size_t)hp.table_floats * 4); }
size_t states_bytes_per_state(const HostPlan &hp) { return (size_t)hp.n_key_slots * 4 + (size_t)hp.ws_floats_per_state * 4; }

}  // namespace

extern "C" {

const char *tqc_last_error(void) { return g_err.c_str(); }
const char *tqc_version(void) { return "tqc-b200 0.1 (sm_100a)"; }

namespace {
// the network without the sliced cuts: kept cuts renumbered in order, axis lists filtered
struct ReducedNet {
    std::vector<int32_t> up, down, ofs, flat;
    std::vector<std::vector<int>> full_axis;
    std::vector<std::vector<std::pair<int, int>>> sliced_axis;
    std::vector<int> c_full, d_extra;
};
bool reduce_network(const tqc_network_desc *net, const int32_t *slice_cuts, int ns, ReducedNet &rn, std::string &why) {
    if (net->m < 1 || net->K < 0 || !net->sub_cut_ofs || (net->K > 0 && (!net->cut_up || !net->cut_down || !net->sub_cuts))) {
        why = "bad network description"; return false;
    }
    std::vector<int> relabel(net->K, 0), is_sliced(net->K, -1);
    for (int i = 0; i < ns; ++i) {
        const int e = slice_cuts[i];
        if (e < 0 || e >= net->K || is_sliced[e] >= 0) { why = "slice_cuts must be distinct cut ids"; return false; }
        is_sliced[e] = i;
    }
    rn.ofs.assign(1, 0);
    for (int e = 0; e < net->K; ++e)
        if (is_sliced[e] < 0) { relabel[e] = (int)rn.up.size(); rn.up.push_back(net->cut_up[e]); rn.down.push_back(net->cut_down[e]); }
    rn.full_axis.assign(net->m, {}); rn.sliced_axis.assign(net->m, {});
    rn.c_full.assign(net->m, 0); rn.d_extra.assign(net->m, 0);
    for (int s = 0; s < net->m; ++s) {
        const int b = net->sub_cut_ofs[s], e1 = net->sub_cut_ofs[s + 1];
        rn.c_full[s] = e1 - b;
        for (int x = b; x < e1; ++x) {
            const int e = net->sub_cuts[x];
            if (e < 0 || e >= net->K) { why = "cut id out of range in sub_cuts"; return false; }
            if (is_sliced[e] >= 0) {
                rn.sliced_axis[s].emplace_back(x - b, is_sliced[e]);
                if (net->cut_down[e] == s) rn.d_extra[s]++;
            } else { rn.flat.push_back(relabel[e]); rn.full_axis[s].push_back(x - b); }
        }
        // local slice digits in the order of slice_cuts (first = most significant)
        std::sort(rn.sliced_axis[s].begin(), rn.sliced_axis[s].end(),
                  [](const std::pair<int, int> &a, const std::pair<int, int> &b2) { return a.second < b2.second; });
        rn.ofs.push_back((int32_t)rn.flat.size());
    }
    return true;
}
void plan_options_from(const tqc_plan_opts *opts, tqc::PlanOptions &po) {
    if (!opts) return;
    po.mode = opts->mode;
    po.restarts = opts->restarts;
    po.seed = opts->seed;
    po.batch_hint = opts->batch_hint;
    po.table_log2_floats_max = opts->table_log2_floats_max;
    po.kmax_cap = opts->kmax_cap;
    po.objective = opts->objective;
    for (int i = 0; i < opts->n_order_steps && opts->order; ++i) po.order.emplace_back(opts->order[2 * i], opts->order[2 * i + 1]);
}
}  // namespace

// Which cuts to slice (the two-level strategy).  Level 1: while a subcircuit tensor of a single
// sub-network, 4^{c'_s} 2^{o_s} floats, exceeds 2^{max_log2_input_floats}, slice "the most size-reducing cut edge": among
// the cuts incident on an oversize tensor the one whose two tensors are largest (compare the larger, then the smaller;
// tie: smaller cut id).  Level 2: while the largest intermediate of the plan exceeds 2^{max_log2_intermediate_floats}
// (4^{open cuts} floats per state; x 2^{carried bits} in distribution mode), slice the cut whose removal gives the smallest
// largest-intermediate, then the smallest total multiplication count, then the smaller id (one greedy plan per candidate).
int tqc_choose_slice_cuts(const tqc_network_desc *net, const tqc_plan_opts *opts, int max_log2_input_floats,
                          int max_log2_intermediate_floats, int32_t *slice_cuts, int32_t *n_slice_cuts) {
    if (!net || !slice_cuts || !n_slice_cuts) return fail(TQC_E_ARG, "null argument");
    {   // the whole description first: level 1 indexes the cut ends, reduce_network only looks at sub_cuts
        std::string verr;
        const int vrc = tqc::validate_network(net->n_qubits, net->m, net->K, net->cut_up, net->cut_down, net->sub_cut_ofs, net->sub_cuts,
                                              net->sub_qubit_ofs, net->sub_qubits, verr);
        if (vrc) return fail(vrc, verr);
    }
    tqc::PlanOptions po;
    plan_options_from(opts, po);
    po.order.clear();                                   // an explicit order names nodes of one particular network
    std::vector<int32_t> S;
    std::vector<char> used(std::max(net->K, 0), 0);
    auto sizes = [&](std::vector<int> &lg) -> bool {
        ReducedNet rn; std::string why;
        if (!reduce_network(net, S.data(), (int)S.size(), rn, why)) { fail(TQC_E_ARG, why); return false; }
        lg.assign(net->m, 0);
        for (int s = 0; s < net->m; ++s)
            lg[s] = 2 * (rn.ofs[s + 1] - rn.ofs[s]) + (net->sub_qubit_ofs ? net->sub_qubit_ofs[s + 1] - net->sub_qubit_ofs[s] : 0);
        return true;
    };
    for (;;) {                                          // level 1: inputs
        std::vector<int> lg;
        if (!sizes(lg)) return TQC_E_ARG;
        if (*std::max_element(lg.begin(), lg.end()) <= max_log2_input_floats) break;
        int best = -1, bhi = -1, blo = -1;
        for (int e = 0; e < net->K; ++e) {
            if (used[e]) continue;
            const int a = lg[net->cut_up[e]], b = lg[net->cut_down[e]];
            if (std::max(a, b) <= max_log2_input_floats) continue;
            const int hi = std::max(a, b), lo = std::min(a, b);
            if (hi > bhi || (hi == bhi && lo > blo)) { best = e; bhi = hi; blo = lo; }
        }
        if (best < 0) return fail(TQC_E_INFEASIBLE, "a subcircuit tensor exceeds max_log2_input_floats with every incident cut sliced");
        used[best] = 1; S.push_back(best);
    }
    struct Score { int max_inter; unsigned __int128 cost; };
    auto score = [&](const std::vector<int32_t> &cuts, Score &sc) -> int {
        ReducedNet rn; std::string why;
        if (!reduce_network(net, cuts.data(), (int)cuts.size(), rn, why)) return fail(TQC_E_ARG, why);
        tqc::HostPlan hp; std::string err;
        const int rc = tqc::build_plan(net->n_qubits, net->m, (int)rn.up.size(), rn.up.data(), rn.down.data(), rn.ofs.data(),
                                       rn.flat.data(), net->sub_qubit_ofs, net->sub_qubits, po, hp, err);
        if (rc) return fail(rc, err);
        sc.max_inter = 0; sc.cost = 0;
        for (int t = 0; t < hp.m - 1; ++t) {
            const Node &C = hp.nodes[hp.m + t];
            sc.max_inter = std::max(sc.max_inter, 2 * (int)C.open.size() + (hp.mode == TQC_MODE_DISTRIBUTION ? (int)C.qubits.size() : 0));
            sc.cost += (unsigned __int128)1 << std::min(hp.steps[t].log2cost, 120);
        }
        return 0;
    };
    for (;;) {                                          // level 2: intermediates
        Score cur;
        int rc = score(S, cur);
        if (rc) return rc;
        if (cur.max_inter <= max_log2_intermediate_floats) break;
        int best = -1; Score bs{0, 0};
        for (int e = 0; e < net->K; ++e) {
            if (used[e]) continue;
            std::vector<int32_t> T = S; T.push_back(e);
            Score sc;
            if ((rc = score(T, sc))) return rc;
            if (best < 0 || sc.max_inter < bs.max_inter || (sc.max_inter == bs.max_inter && sc.cost < bs.cost)) { best = e; bs = sc; }
        }
        if (best < 0) return fail(TQC_E_INFEASIBLE, "an intermediate exceeds max_log2_intermediate_floats with every cut sliced");
        used[best] = 1; S.push_back(best);
    }
    for (size_t i = 0; i < S.size(); ++i) slice_cuts[i] = S[i];
    *n_slice_cuts = (int32_t)S.size();
    return 0;
}

int tqc_plan(const tqc_network_desc *net, const tqc_plan_opts *opts, tqc_plan_t **out) {
    if (!net || !out) return fail(TQC_E_ARG, "null argument");
    tqc::PlanOptions po;
    int use_tc = 0;
    if (opts) {
        po.mode = opts->mode;
        po.restarts = opts->restarts;
        po.seed = opts->seed;
        po.batch_hint = opts->batch_hint;
        po.table_log2_floats_max = opts->table_log2_floats_max;
        po.kmax_cap = opts->kmax_cap;
        po.objective = opts->objective;
        use_tc = opts->use_tcgen05;
        if (opts->n_order_steps > 0) {
            if (!opts->order) return fail(TQC_E_ARG, "n_order_steps > 0 but order is null");
            for (int i = 0; i < opts->n_order_steps; ++i) po.order.emplace_back(opts->order[2 * i], opts->order[2 * i + 1]);
        }
    }
    tqc_plan_t *pl = new tqc_plan_t();
    std::string err;
    int rc;
    const int ns = opts ? opts->n_slice_cuts : 0;
    if (ns < 0 || (ns > 0 && !opts->slice_cuts)) { delete pl; return fail(TQC_E_ARG, "n_slice_cuts > 0 but slice_cuts is null"); }
    if (ns > 12) { delete pl; return fail(TQC_E_TOO_LARGE, "at most 12 sliced cuts (4^12 sub-networks)"); }
    pl->K_full = net->K;
    if (ns == 0) {
        rc = tqc::build_plan(net->n_qubits, net->m, net->K, net->cut_up, net->cut_down, net->sub_cut_ofs,
                             net->sub_cuts, net->sub_qubit_ofs, net->sub_qubits, po, pl->hp, err);
    } else {
        // the planner only sees the reduced network: check the caller's whole description here (ends of the sliced cuts,
        // each cut listed by exactly its two subcircuits), else a malformed sliced cut would silently give a wrong sum
        std::string verr;
        const int vrc = tqc::validate_network(net->n_qubits, net->m, net->K, net->cut_up, net->cut_down, net->sub_cut_ofs, net->sub_cuts,
                                              net->sub_qubit_ofs, net->sub_qubits, verr);
        if (vrc) { delete pl; return fail(vrc, verr); }
        ReducedNet rn;
        std::string why;
        if (!reduce_network(net, opts->slice_cuts, ns, rn, why)) { delete pl; return fail(TQC_E_ARG, why); }
        pl->slice_cuts.assign(opts->slice_cuts, opts->slice_cuts + ns);
        pl->full_axis = rn.full_axis; pl->sliced_axis = rn.sliced_axis; pl->c_full = rn.c_full; pl->d_extra = rn.d_extra;
        const std::vector<int32_t> &up = rn.up, &down = rn.down, &ofs = rn.ofs, &flat = rn.flat;
        rc = tqc::build_plan(net->n_qubits, net->m, (int)up.size(), up.data(), down.data(), ofs.data(), flat.data(),
                             net->sub_qubit_ofs, net->sub_qubits, po, pl->hp, err);
    }
    if (rc != 0) { delete pl; return fail(rc, err); }
    pl->use_tcgen05 = use_tc;
    pl->plan_opts = po;
    pl->d_leaf_all.assign(pl->hp.m, nullptr);
    pl->d_leaf.assign(pl->hp.m, nullptr);
    pl->loaded.assign(pl->hp.m, 0);
    for (int t = 0; t < pl->hp.m - 1; ++t) {
        Step &s = pl->hp.steps[t];
        const bool batch = pl->hp.nodes[pl->hp.m + t].kind == tqc::NODE_BATCH;
        s.kernel_class = (s.outer_lhs.empty() && s.outer_rhs.empty() && batch) ? TQC_KERNEL_DOT : TQC_KERNEL_SIMT_TILE;
        if (batch && use_tc >= 0 && tc_eligible(2 * (int)s.outer_lhs.size(), 2 * (int)s.outer_rhs.size(), 2 * (int)s.inner.size()))
            s.kernel_class = TQC_KERNEL_TCGEN05;
    }
    pl->chain_mode = opts ? opts->use_chain : 0;
    if (pl->n_sliced()) pl->chain_mode = -1;                // the chain's device step table holds leaf pointers; sliced plans run per step
    pl->chain = pl->chain_mode != -1 && build_chain(pl);
    if (pl->chain) pl->hp.ws_floats_per_state = 0;          // intermediates live in shared memory
    if (pl->chain) {
        if (const char *dump = dev_env("TQC_CHAIN_SRC_DUMP")) {      // development aid: the generated specialisation
            if (FILE *f = fopen(dump, "w")) { fputs(chain_source(pl).c_str(), f); fclose(f); }
        }
    }
    if (pl->chain)
        for (int t = 0; t < pl->hp.m - 1; ++t)
            if (pl->hp.nodes[pl->hp.m + t].kind == tqc::NODE_BATCH) pl->hp.steps[t].kernel_class = TQC_KERNEL_CHAIN;
    *out = pl;
    return 0;
}

void tqc_plan_destroy(tqc_plan_t *pl) {
    if (!pl) return;
    for (size_t x = 0; x < pl->d_leaf.size(); ++x) {
        float *p = pl->n_sliced() ? pl->d_leaf_all[x] : pl->d_leaf[x];
        if (p) cudaFree(p);
    }
    if (pl->d_slot_ofs) cudaFree(pl->d_slot_ofs);
    if (pl->d_slot_qubits) cudaFree(pl->d_slot_qubits);
    if (pl->d_staging) cudaFree(pl->d_staging);
    if (pl->d_chain) cudaFree(pl->d_chain);
    if (pl->jit_module && jit_api().ok) jit_api().ModuleUnload((CUmodule)pl->jit_module);
    for (cudaEvent_t e : pl->ev_pool) cudaEventDestroy(e);
    if (pl->hss_sub) tqc_plan_destroy(pl->hss_sub);
    delete pl->cut;
    if (pl->ev_fork) cudaEventDestroy(pl->ev_fork);
    for (int l = 0; l < tqc_plan::N_LANES; ++l) {
        if (pl->ev_join[l]) cudaEventDestroy(pl->ev_join[l]);
        if (pl->lane[l]) { cudaStreamSynchronize(pl->lane[l]); cudaStreamDestroy(pl->lane[l]); }
    }
    delete pl;
}

int tqc_plan_mode(const tqc_plan_t *pl) { return pl ? pl->hp.mode : TQC_E_ARG; }
int tqc_plan_num_qubits(const tqc_plan_t *pl) { return pl ? pl->hp.n : TQC_E_ARG; }
int tqc_plan_num_subcircuits(const tqc_plan_t *pl) { return pl ? pl->hp.m : TQC_E_ARG; }
int tqc_plan_num_cuts(const tqc_plan_t *pl) { return pl ? pl->K_full : TQC_E_ARG; }
int tqc_plan_num_sliced_cuts(const tqc_plan_t *pl) { return pl ? pl->n_sliced() : TQC_E_ARG; }
int tqc_plan_num_steps(const tqc_plan_t *pl) { return pl ? (int)pl->hp.steps.size() : TQC_E_ARG; }
int tqc_plan_kmax(const tqc_plan_t *pl) { return pl ? pl->hp.kmax : TQC_E_ARG; }

int tqc_plan_tensor_shape(const tqc_plan_t *pl, int s, int *c_s, int *o_s) {
    if (!pl || s < 0 || s >= pl->hp.m) return fail(TQC_E_ARG, "bad plan or subcircuit id");
    if (c_s) *c_s = pl->n_sliced() ? pl->c_full[s] : pl->hp.c(s);
    if (o_s) *o_s = pl->hp.o(s);
    return 0;
}

int tqc_plan_step(const tqc_plan_t *pl, int i, int *lhs, int *rhs, int *n_inner, int *n_outer_lhs, int *n_outer_rhs,
                  int *log2cost, int *kernel_class) {
    if (!pl || i < 0 || i >= (int)pl->hp.steps.size()) return fail(TQC_E_ARG, "bad plan or step id");
    const Step &s = pl->hp.steps[i];
    if (lhs) *lhs = s.lhs;
    if (rhs) *rhs = s.rhs;
    if (n_inner) *n_inner = (int)s.inner.size();
    if (n_outer_lhs) *n_outer_lhs = (int)s.outer_lhs.size();
    if (n_outer_rhs) *n_outer_rhs = (int)s.outer_rhs.size();
    if (log2cost) *log2cost = s.log2cost;
    if (kernel_class) *kernel_class = s.kernel_class;
    return 0;
}

int tqc_plan_node(const tqc_plan_t *pl, int v, int *kind, int *n_bits, int *n_open) {
    if (!pl || v < 0 || v >= (int)pl->hp.nodes.size()) return fail(TQC_E_ARG, "bad plan or node id");
    const Node &nd = pl->hp.nodes[v];
    if (kind) *kind = nd.kind;
    if (n_bits) *n_bits = (int)nd.qubits.size();
    if (n_open) *n_open = (int)nd.open.size();
    return 0;
}

double tqc_plan_cost_log2(const tqc_plan_t *pl) { return pl ? tqc::cost_log2(pl->hp) : -1.0; }
double tqc_plan_modelled_seconds_per_state(const tqc_plan_t *pl) {
    if (!pl || pl->hp.mode != TQC_MODE_STATES) return -1.0;
    return (double)tqc::plan_time_fs(pl->hp, pl->plan_opts) * 1e-15 * std::ldexp(1.0, 2 * pl->n_sliced());
}

int tqc_plan_serialize(const tqc_plan_t *pl, void *buf, size_t *len) {
    if (!pl || !len) return fail(TQC_E_ARG, "null argument");
    const std::vector<int32_t> w = tqc::serialize_words(pl->hp);
    const size_t need = 8 + w.size() * 4;
    if (!buf) { *len = need; return 0; }
    if (*len < need) { *len = need; return fail(TQC_E_ARG, "buffer too small"); }
    unsigned char *b = (unsigned char *)buf;
    memcpy(b, "TQCP", 4);
    const int32_t version = 1;
    memcpy(b + 4, &version, 4);
    memcpy(b + 8, w.data(), w.size() * 4);
    *len = need;
    return 0;
}

size_t tqc_plan_workspace_min_bytes(const tqc_plan_t *pl) {
    if (!pl) return 0;
    if (pl->hp.mode == TQC_MODE_STATES)
        return states_fixed_bytes(pl->hp) + align256(states_bytes_per_state(pl->hp) * 64) + 256 + (pl->n_sliced() ? 1024 : 0);
    return tqc_plan_workspace_bytes(pl, 0, 0);
}

size_t tqc_plan_workspace_bytes(const tqc_plan_t *pl, size_t n_states, int prefix_bits) {
    if (!pl) return 0;
    const HostPlan &hp = pl->hp;
    if (hp.mode == TQC_MODE_STATES) {
        const size_t cap = (std::max<size_t>(n_states, 1) + 63) / 64 * 64;
        return states_fixed_bytes(hp) + align256(states_bytes_per_state(hp) * cap) + 256 + (pl->n_sliced() ? align256(n_states * 4) : 0);
    }
    std::vector<int> fb;
    std::vector<int64_t> off;
    const int pbits = std::max(0, std::min(prefix_bits, hp.n));
    const int64_t floats = tqc::distribution_layout(hp, pbits, fb, off);
    return align256((size_t)floats * 4) + 256 + (pl->n_sliced() ? align256(((size_t)4) << (hp.n - pbits)) : 0);
}

int tqc_load_subcircuit_tensors(tqc_plan_t *pl, int s, const float *data, size_t n_elems, int on_device, void *stream) {
    if (!pl || !data) return fail(TQC_E_ARG, "null argument");
    HostPlan &hp = pl->hp;
    if (s < 0 || s >= hp.m) return fail(TQC_E_ARG, "subcircuit id out of range");
    const bool sliced = pl->n_sliced() > 0;
    const int c = hp.c(s), o = hp.o(s);                     // c: axes the plan contracts (without the sliced ones)
    const int cf = sliced ? pl->c_full[s] : c;              // axes of the caller's tensor
    const int nsl = sliced ? (int)pl->sliced_axis[s].size() : 0;
    const size_t need = (size_t)1 << (2 * cf + o);
    if (n_elems != need) return fail(TQC_E_SHAPE, "n_elems must be 4^c_s * 2^o_s = " + std::to_string(need));
    cudaStream_t st = (cudaStream_t)stream;
    int rc = ensure_device_attrs(&pl->sm_count);
    if (rc) return rc;
    float *&store = sliced ? pl->d_leaf_all[s] : pl->d_leaf[s];
    if (!store) TQC_CUDA(cudaMalloc(&store, need * sizeof(float)));
    if (sliced) pl->d_leaf[s] = store;
    const float *src = data;
    if (!on_device) {
        if (pl->staging_elems < need) {
            if (pl->d_staging) { TQC_CUDA(cudaStreamSynchronize(st)); TQC_CUDA(cudaFree(pl->d_staging)); pl->d_staging = nullptr; }
            TQC_CUDA(cudaMalloc(&pl->d_staging, need * sizeof(float)));
            pl->staging_elems = need;
        }
        TQC_CUDA(cudaMemcpyAsync(pl->d_staging, data, need * sizeof(float), cudaMemcpyHostToDevice, st));
        src = pl->d_staging;
    }
    RelayoutArgs a;
    memset(&a, 0, sizeof(a));
    a.src = src;
    a.lgRows = 2 * c; a.lgCols = o;
    // 2^{-d_s}: one factor 1/2 per cut whose downstream end is s (reading G2), the sliced ones included
    a.scale = std::ldexp(1.0f, -(hp.d[s] + (sliced ? pl->d_extra[s] : 0)));
    // device digit x (most significant first) holds cut layout[x]; the caller's digit order is sub_cuts[s]
    const Node &leaf = hp.nodes[s];
    std::vector<int> layout = leaf.layout;
    if (layout.empty()) layout = leaf.open;               // m == 1 has no consumer: keep ascending order
    BitPairs bp;
    for (int x = 0; x < c; ++x) {
        const int y = index_of(hp.sub_cuts[s], layout[x]);            // position among the kept axes
        const int yf = sliced ? pl->full_axis[s][y] : y;              // position among the caller's axes
        bp.add_run(2 * (c - 1 - x), 2 * (cf - 1 - yf), 2);
    }
    if (!bp.build(a.row_of)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
    const long long tiles = (((1ll << o) + 31) / 32) * (((1ll << (2 * c)) + 31) / 32);
    const bool prof = pl->profile;
    pl->profile = false;                                   // loads are not part of the profiled contract call
    // one re-laid-out sub-tensor per value of the sliced axes (a single one without slicing)
    for (long long v = 0; v < (1ll << (2 * nsl)); ++v) {
        a.dst = store + (size_t)v * ((size_t)1 << (2 * c + o));
        a.row_or = 0;
        for (int x = 0; x < nsl; ++x) {                                // local digit x, first = most significant
            const unsigned long long digit = (unsigned long long)(v >> (2 * (nsl - 1 - x))) & 3ull;
            a.row_or |= digit << (2 * (cf - 1 - pl->sliced_axis[s][x].first));
        }
        rc = note_launch(pl, TAG_RELAYOUT, st);
        if (rc) break;
        tqc::relayout_kernel<<<(unsigned)tiles, 256, 0, st>>>(a);
    }
    pl->profile = prof;
    if (rc) return rc;
    TQC_CUDA(cudaGetLastError());
    pl->loaded[s] = 1;
    // the load that completes the tensor set also prepares the plan for the contract calls (a reload keeps the same
    // device allocation, so a finalized plan stays valid)
    if (!pl->finalized && std::all_of(pl->loaded.begin(), pl->loaded.end(), [](char c) { return c != 0; })) return tqc_plan_finalize(pl, stream);
    return 0;
}

// Everything a contract call needs beyond the tensors, done ONCE here so that the contract calls neither allocate nor
// synchronise: kernel attributes of this device, the key-slot tables, the device step table of the fused chain and its
// plan-specialised kernel (NVRTC compile + module load), the side streams and events of the forked table steps.
int tqc_plan_finalize(tqc_plan_t *pl, void *stream) {
    (void)stream;
    if (!pl) return fail(TQC_E_ARG, "null plan");
    for (int s = 0; s < pl->hp.m; ++s) if (!pl->loaded[s]) return fail(TQC_E_STATE, "tensor of subcircuit " + std::to_string(s) + " not loaded");
    if (pl->finalized) return 0;
    int rc;
    if ((rc = ensure_device_attrs(&pl->sm_count))) return rc;
    if ((rc = ensure_meta(pl))) return rc;
    if ((rc = ensure_chain(pl))) return rc;
    if ((rc = ensure_lanes(pl))) return rc;
    pl->finalized = true;
    return 0;
}

namespace {
// point every leaf at the sub-tensor of slice assignment `assign` (base-4 digits in the order of slice_cuts, first = MS)
void select_slice(tqc_plan_t *pl, long long assign) {
    const int ns = pl->n_sliced();
    for (int s = 0; s < pl->hp.m; ++s) {
        if (!pl->d_leaf_all[s]) continue;
        size_t local = 0;
        for (const auto &ax : pl->sliced_axis[s]) local = local * 4 + (size_t)((assign >> (2 * (ns - 1 - ax.second))) & 3);
        pl->d_leaf[s] = pl->d_leaf_all[s] + local * ((size_t)1 << (2 * pl->hp.c(s) + pl->hp.o(s)));
    }
}
int contract_states_impl(tqc_plan_t *pl, const uint64_t *states_dev, size_t n_states, float *out_dev, void *workspace_dev,
                         size_t workspace_bytes, void *stream, bool fork_recorded = false);
int contract_distribution_impl(tqc_plan_t *pl, uint64_t prefix_value, int prefix_bits, float *out_dev, void *workspace_dev,
                               size_t workspace_bytes, void *stream);
// sum over the 4^{n_sliced} sub-networks: the first lands in out, the others in a partial-sum buffer at the head of the
// workspace and are added ("a summation of smaller tensor networks")
int sliced_sum(tqc_plan_t *pl, float *out_dev, size_t n_out, void *workspace_dev, size_t workspace_bytes, void *stream,
               const std::function<int(float *, void *, size_t)> &once) {
    if (!workspace_dev || ((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be non-null and 256-byte aligned");
    const size_t tb = align256(n_out * 4);
    if (workspace_bytes < tb) return fail(TQC_E_WORKSPACE, "workspace smaller than the partial-sum buffer of a sliced plan");
    float *tmp = (float *)workspace_dev;
    char *rest = (char *)workspace_dev + tb;
    cudaStream_t st = (cudaStream_t)stream;
    int rc = 0;
    for (long long a = 0; a < (1ll << (2 * pl->n_sliced())) && !rc; ++a) {
        select_slice(pl, a);
        rc = once(a == 0 ? out_dev : tmp, rest, workspace_bytes - tb);
        if (!rc && a > 0) {
            pl->launches++;
            tqc::accumulate_kernel<<<(unsigned)std::min<size_t>((n_out + 1023) / 1024, 148 * 16), 256, 0, st>>>(out_dev, tmp, (long long)n_out);
            if (cudaGetLastError() != cudaSuccess) rc = fail(TQC_E_CUDA, "accumulate_kernel launch failed");
        }
    }
    select_slice(pl, 0);
    return rc;
}
}  // namespace

int tqc_contract_states(tqc_plan_t *pl, const uint64_t *states_dev, size_t n_states, float *out_dev, void *workspace_dev,
                        size_t workspace_bytes, void *stream) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    if (pl->n_sliced() == 0 || n_states == 0) return contract_states_impl(pl, states_dev, n_states, out_dev, workspace_dev, workspace_bytes, stream);
    if (!out_dev || !states_dev) return fail(TQC_E_ARG, "null states/out pointer");
    // the partial-sum buffer (4 bytes per state) comes out of the workspace: when it does not fit for the whole batch next to
    // the plan's own minimum, the batch is cut into pieces of `piece` states, each summed over all sub-networks
    const size_t fixed = states_fixed_bytes(pl->hp), per = states_bytes_per_state(pl->hp) + 4;
    if (workspace_bytes < fixed + 1024 + per * 64) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_plan_workspace_min_bytes");
    size_t piece = (workspace_bytes - fixed - 1024) / per / 64 * 64;
    piece = std::min(piece, (n_states + 63) / 64 * 64);
    const size_t words = (size_t)(pl->hp.n + 63) / 64;
    for (size_t lo = 0; lo < n_states; lo += piece) {
        const size_t cnt = std::min(piece, n_states - lo);
        const int rc = sliced_sum(pl, out_dev + lo, cnt, workspace_dev, workspace_bytes, stream, [&](float *dst, void *ws, size_t wb) {
            return contract_states_impl(pl, states_dev + lo * words, cnt, dst, ws, wb, stream);
        });
        if (rc) return rc;
    }
    return 0;
}

int tqc_contract_distribution(tqc_plan_t *pl, uint64_t prefix_value, int prefix_bits, float *out_dev, void *workspace_dev,
                              size_t workspace_bytes, void *stream) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    if (pl->n_sliced() == 0) return contract_distribution_impl(pl, prefix_value, prefix_bits, out_dev, workspace_dev, workspace_bytes, stream);
    if (!out_dev) return fail(TQC_E_ARG, "null out pointer");
    if (prefix_bits < 0 || prefix_bits > pl->hp.n) return fail(TQC_E_ARG, "prefix_bits out of range");
    if (pl->hp.n - prefix_bits > 34) return fail(TQC_E_TOO_LARGE, "more than 2^34 outputs; raise prefix_bits");
    return sliced_sum(pl, out_dev, (size_t)1 << (pl->hp.n - prefix_bits), workspace_dev, workspace_bytes, stream,
                      [&](float *dst, void *ws, size_t wb) { return contract_distribution_impl(pl, prefix_value, prefix_bits, dst, ws, wb, stream); });
}

namespace {
// fork_recorded: the caller (host-buffer entry point) has already recorded ev_fork on the stream, before its H2D copy
int contract_states_impl(tqc_plan_t *pl, const uint64_t *states_dev, size_t n_states, float *out_dev, void *workspace_dev,
                        size_t workspace_bytes, void *stream, bool fork_recorded) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    HostPlan &hp = pl->hp;
    if (hp.mode != TQC_MODE_STATES) return fail(TQC_E_STATE, "plan was built for distribution mode");
    for (int s = 0; s < hp.m; ++s) if (!pl->loaded[s]) return fail(TQC_E_STATE, "tensor of subcircuit " + std::to_string(s) + " not loaded");
    if (n_states == 0) return 0;
    if (!states_dev || !out_dev) return fail(TQC_E_ARG, "null states/out pointer");
    if (n_states > (size_t)0x7fffffff) return fail(TQC_E_TOO_LARGE, "more than 2^31-1 states in one call");
    cudaStream_t st = (cudaStream_t)stream;
    const size_t fixed = states_fixed_bytes(hp), per = states_bytes_per_state(hp);
    if ((fixed + per > 0) && !workspace_dev) return fail(TQC_E_WORKSPACE, "workspace is null");
    if (((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be 256-byte aligned");
    long long cap;
    if (per == 0) cap = (long long)((n_states + 63) / 64 * 64);
    else {
        if (workspace_bytes < fixed + 256) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_plan_workspace_min_bytes");
        cap = (long long)((workspace_bytes - fixed - 256) / per) / 64 * 64;
        cap = std::min<long long>(cap, (long long)((n_states + 63) / 64 * 64));
        if (cap < 64) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_plan_workspace_min_bytes");
    }
    char *ws = (char *)workspace_dev;
    float *tables = (float *)ws;
    uint32_t *keys = (uint32_t *)(ws + fixed);
    float *batch = (float *)(ws + fixed + align256((size_t)hp.n_key_slots * 4 * (size_t)cap));
    // the alignment pad of the key region is covered by the +256 of tqc_plan_workspace_bytes
    int rc;
    if (!pl->finalized) return fail(TQC_E_STATE, "plan not finalized (tqc_plan_finalize runs at the last tqc_load_subcircuit_tensors)");
    prof_begin(pl);
    // phase T: nodes evaluated once per key (tables), independent of the batch
    CrossCtx cx;
    cx.ws = tables;
    // Table steps whose operands are all leaves neither depend on one another nor share storage (plan.cpp releases a
    // table's block only when another table step consumes it): they go to side streams and overlap the key kernel.
    const bool fork = pl->tables_parallel == 1 && !pl->profile;
    int lanes_used = 0;
    if (fork) {
        if (!fork_recorded) TQC_CUDA(cudaEventRecord(pl->ev_fork, st));
        int next = 0;
        for (int t = 0; t < hp.m - 1; ++t) {
            if (hp.nodes[hp.m + t].kind != tqc::NODE_TABLE) continue;
            const int l = next++ % tqc_plan::N_LANES;
            if (l >= lanes_used) { TQC_CUDA(cudaStreamWaitEvent(pl->lane[l], pl->ev_fork, 0)); lanes_used = l + 1; }
            if ((rc = launch_cross_step(pl, cx, t, pl->lane[l]))) return rc;
        }
        for (int l = 0; l < lanes_used; ++l) TQC_CUDA(cudaEventRecord(pl->ev_join[l], pl->lane[l]));
    } else
    for (int t = 0; t < hp.m - 1; ++t)
        if (hp.nodes[hp.m + t].kind == tqc::NODE_TABLE && (rc = launch_cross_step(pl, cx, t, st))) return rc;
    // phase B: chunks of states
    const int words = (hp.n + 63) / 64;
    const Node &root = hp.nodes[hp.root()];
    for (size_t lo = 0; lo < n_states; lo += (size_t)cap) {
        BatchCtx bx;
        bx.tables = tables; bx.keys = keys; bx.batch = batch; bx.cap = cap;
        bx.R = (int)std::min<size_t>((size_t)cap, n_states - lo);
        bx.out = out_dev + lo;
        if (hp.n_key_slots > 0) {
            KeyArgs ka;
            ka.states = states_dev + lo * (size_t)std::max(words, 0);
            ka.keys = keys; ka.slot_ofs = pl->d_slot_ofs; ka.slot_qubits = pl->d_slot_qubits;
            ka.words = words; ka.R = bx.R; ka.cap = cap;
            dim3 grid((unsigned)((bx.R + 255) / 256), (unsigned)hp.n_key_slots);
            if ((rc = note_launch(pl, TAG_KEYS, st))) return rc;
            tqc::key_kernel<<<grid, 256, 0, st>>>(ka);
            TQC_CUDA(cudaGetLastError());
        }
        if (lo == 0) for (int l = 0; l < lanes_used; ++l) TQC_CUDA(cudaStreamWaitEvent(st, pl->ev_join[l], 0));   // join
        if (pl->chain) {
            tqc::ChainArgs ca;
            memset(&ca, 0, sizeof(ca));
            ca.steps = pl->d_chain; ca.n_steps = (int)pl->chain_host.size();
            ca.tables = tables; ca.keys = keys; ca.cap = cap; ca.out = bx.out; ca.R = bx.R;
            ca.scratch_floats = pl->chain_scratch; ca.stage_floats = pl->chain_stage;
            ca.n_slots = hp.n_key_slots;
            ca.n_gather = (int)pl->chain_gather.size(); ca.total_f4 = pl->chain_f4; ca.tab_entries = pl->chain_tab_entries;
            for (int x = 0; x < ca.n_gather; ++x) {
                ca.g[x] = pl->chain_gather[x];
                if (pl->chain_gather_leaf[x] >= 0) ca.g[x].base = pl->d_leaf[pl->chain_gather_leaf[x]];
            }
            const size_t smem = (((size_t)ca.n_steps * sizeof(tqc::ChainStep) + 15) & ~(size_t)15) +
                                (((size_t)ca.tab_entries * 2 + 15) & ~(size_t)15) + (size_t)ca.total_f4 * 16 +
                                (size_t)tqc::CHAIN_WARPS * pl->chain_scratch * 4;
            const long long blocks = std::min<long long>((bx.R + tqc::CHAIN_WARPS - 1) / tqc::CHAIN_WARPS, 148ll * 8);
            if ((rc = note_launch(pl, TAG_CHAIN, st))) return rc;
            if (pl->jit_fn) {
                void *params[] = {&ca};
                const CUresult lr = jit_api().LaunchKernel((CUfunction)pl->jit_fn, (unsigned)blocks, 1, 1, tqc::CHAIN_WARPS * 32, 1, 1,
                                                           (unsigned)smem, (CUstream)st, params, nullptr);
                if (lr != CUDA_SUCCESS) return fail(TQC_E_CUDA, "cuLaunchKernel(chain_spec_kernel) failed with code " + std::to_string((int)lr));
            } else
            tqc::chain_kernel<<<(unsigned)blocks, tqc::CHAIN_WARPS * 32, smem, st>>>(ca);
            TQC_CUDA(cudaGetLastError());
        } else
        for (int t = 0; t < hp.m - 1; ++t)
            if (hp.nodes[hp.m + t].kind == tqc::NODE_BATCH && (rc = launch_batch_step(pl, bx, t, st))) return rc;
        if (root.kind != tqc::NODE_BATCH) {
            GatherArgs g;
            memset(&g, 0, sizeof(g));
            g.table = hp.m == 1 ? pl->d_leaf[0] : tables + root.table_offset;
            g.keys = keys + (long long)root.key_slot * cap;
            g.out = bx.out; g.R = bx.R;
            if ((rc = note_launch(pl, TAG_GATHER, st))) return rc;
            tqc::gather_kernel<<<(unsigned)((bx.R + 255) / 256), 256, 0, st>>>(g);
            TQC_CUDA(cudaGetLastError());
        }
    }
    return prof_close(pl, st);
}

int contract_distribution_impl(tqc_plan_t *pl, uint64_t prefix_value, int prefix_bits, float *out_dev, void *workspace_dev,
                              size_t workspace_bytes, void *stream) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    HostPlan &hp = pl->hp;
    if (hp.mode != TQC_MODE_DISTRIBUTION) return fail(TQC_E_STATE, "plan was built for states mode");
    for (int s = 0; s < hp.m; ++s) if (!pl->loaded[s]) return fail(TQC_E_STATE, "tensor of subcircuit " + std::to_string(s) + " not loaded");
    if (!pl->finalized) return fail(TQC_E_STATE, "plan not finalized (tqc_plan_finalize runs at the last tqc_load_subcircuit_tensors)");
    if (prefix_bits < 0 || prefix_bits > hp.n || prefix_bits > 64) return fail(TQC_E_ARG, "prefix_bits out of range");
    if (prefix_bits < 64 && (prefix_value >> prefix_bits) != 0) return fail(TQC_E_ARG, "prefix_value has more than prefix_bits bits");
    if (hp.n - prefix_bits > 34) return fail(TQC_E_TOO_LARGE, "more than 2^34 outputs; raise prefix_bits");
    if (!out_dev) return fail(TQC_E_ARG, "null out pointer");
    cudaStream_t st = (cudaStream_t)stream;
    std::vector<int> fb;
    std::vector<int64_t> off;
    const int64_t floats = tqc::distribution_layout(hp, prefix_bits, fb, off);
    if (floats > 0) {
        if (!workspace_dev || workspace_bytes < (size_t)floats * 4) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_plan_workspace_bytes");
        if (((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be 256-byte aligned");
    }
    CrossCtx cx;
    cx.prefix_bits = prefix_bits; cx.prefix_value = prefix_value;
    cx.free_bits = &fb; cx.offsets = &off;
    cx.ws = (float *)workspace_dev; cx.out = out_dev;
    int rc;
    prof_begin(pl);
    for (int t = 0; t < hp.m - 1; ++t)
        if ((rc = launch_cross_step(pl, cx, t, st))) return rc;
    if (hp.m == 1) {
        // K = 0: p(x) = T_0[x] (reading G15), permuted from the listed qubit order to global bit order
        const Node &leaf = hp.nodes[0];
        GatherArgs g;
        memset(&g, 0, sizeof(g));
        const std::vector<int> fq = free_qubits(leaf, prefix_bits);
        const int nq = (int)leaf.qubits.size(), nf = (int)fq.size();
        BitPairs in, om;
        unsigned long long fixed = 0;
        int t = 0;
        for (int pq = 0; pq < nq; ++pq) {
            const int q = leaf.qubits[pq];
            if (q >= prefix_bits) {
                int dst = 0;
                for (int x : fq) if (x > q) ++dst;
                in.add(nf - 1 - t, nq - 1 - pq);
                om.add(nf - 1 - t, dst);
                ++t;
            } else if ((prefix_value >> (prefix_bits - 1 - q)) & 1ull) fixed |= 1ull << (nq - 1 - pq);
        }
        if (!in.build(g.map) || !om.build(g.out_map)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
        g.map_or = fixed;
        g.table = pl->d_leaf[0]; g.keys = nullptr; g.out = out_dev; g.R = 1ll << nf;
        if ((rc = note_launch(pl, TAG_GATHER, st))) return rc;
        tqc::gather_kernel<<<(unsigned)((g.R + 255) / 256), 256, 0, st>>>(g);
        TQC_CUDA(cudaGetLastError());
    }
    return prof_close(pl, st);
}
}  // namespace

// ---- host-buffer entry points: staging carved from the front of the workspace ------------------
size_t tqc_plan_workspace_bytes_host(const tqc_plan_t *pl, size_t n_states, int prefix_bits) {
    if (!pl) return 0;
    const HostPlan &hp = pl->hp;
    if (hp.mode == TQC_MODE_STATES) {
        const size_t words = (size_t)(hp.n + 63) / 64;
        return align256(n_states * words * 8) + align256(n_states * 4) + tqc_plan_workspace_bytes(pl, n_states, 0);
    }
    const int pb = std::max(0, std::min(prefix_bits, hp.n));
    return align256(((size_t)4) << (hp.n - pb)) + tqc_plan_workspace_bytes(pl, 0, pb);
}

int tqc_contract_states_host(tqc_plan_t *pl, const uint64_t *states_host, size_t n_states, float *out_host,
                             void *workspace_dev, size_t workspace_bytes, void *stream) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    if (n_states == 0) return 0;
    if (!states_host || !out_host) return fail(TQC_E_ARG, "null states/out pointer");
    if (!workspace_dev || ((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be non-null and 256-byte aligned");
    const size_t words = (size_t)(pl->hp.n + 63) / 64;
    const size_t sb = align256(n_states * words * 8), ob = align256(n_states * 4);
    if (workspace_bytes < sb + ob + tqc_plan_workspace_min_bytes(pl)) return fail(TQC_E_WORKSPACE, "workspace smaller than staging + tqc_plan_workspace_min_bytes");
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace_dev;
    uint64_t *sd = (uint64_t *)ws;
    float *od = (float *)(ws + sb);
    // the table steps do not depend on the states: fork their side streams off BEFORE the host-to-device copy so that
    // they run under it (only for the plain path: a sliced plan loops over sub-networks, profile mode stays serial)
    bool forked = false;
    if (pl->hp.mode == TQC_MODE_STATES && pl->n_sliced() == 0 && !pl->profile && pl->finalized && pl->tables_parallel == 1) {
        TQC_CUDA(cudaEventRecord(pl->ev_fork, st));
        forked = true;
    }
    if (words > 0) TQC_CUDA(cudaMemcpyAsync(sd, states_host, n_states * words * 8, cudaMemcpyHostToDevice, st));
    const int rc = forked ? contract_states_impl(pl, sd, n_states, od, ws + sb + ob, workspace_bytes - sb - ob, stream, true)
                          : tqc_contract_states(pl, sd, n_states, od, ws + sb + ob, workspace_bytes - sb - ob, stream);
    if (rc) return rc;
    TQC_CUDA(cudaMemcpyAsync(out_host, od, n_states * 4, cudaMemcpyDeviceToHost, st));
    return 0;
}

int tqc_contract_distribution_host(tqc_plan_t *pl, uint64_t prefix_value, int prefix_bits, float *out_host,
                                   void *workspace_dev, size_t workspace_bytes, void *stream) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    if (!out_host) return fail(TQC_E_ARG, "null out pointer");
    if (prefix_bits < 0 || prefix_bits > pl->hp.n) return fail(TQC_E_ARG, "prefix_bits out of range");
    if (pl->hp.n - prefix_bits > 34) return fail(TQC_E_TOO_LARGE, "more than 2^34 outputs; raise prefix_bits");
    if (!workspace_dev || ((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be non-null and 256-byte aligned");
    const size_t ob = align256(((size_t)4) << (pl->hp.n - prefix_bits));
    if (workspace_bytes < ob) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_plan_workspace_bytes_host");
    cudaStream_t st = (cudaStream_t)stream;
    char *ws = (char *)workspace_dev;
    const int rc = tqc_contract_distribution(pl, prefix_value, prefix_bits, (float *)ws, ws + ob, workspace_bytes - ob, stream);
    if (rc) return rc;
    TQC_CUDA(cudaMemcpyAsync(out_host, ws, ((size_t)4) << (pl->hp.n - prefix_bits), cudaMemcpyDeviceToHost, st));
    return 0;
}

// ---- per-launch timing --------------------------------------------------------------------------
int tqc_plan_profile_enable(tqc_plan_t *pl, int on) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    pl->profile = on != 0;
    pl->ev_used = 0;
    pl->ev_tags.clear();
    return 0;
}

int tqc_plan_profile_read(tqc_plan_t *pl, int32_t *tags, float *ms, size_t *n) {
    if (!pl || !n) return fail(TQC_E_ARG, "null argument");
    const size_t have = pl->ev_tags.size();
    if (!tags || !ms) { *n = have; return 0; }
    if (*n < have) { *n = have; return fail(TQC_E_ARG, "buffer too small"); }
    if (have > 0) {
        if (pl->ev_used != have + 1) return fail(TQC_E_STATE, "profiled call did not complete");
        TQC_CUDA(cudaEventSynchronize(pl->ev_pool[have]));
        for (size_t i = 0; i < have; ++i) {
            tags[i] = pl->ev_tags[i];
            TQC_CUDA(cudaEventElapsedTime(&ms[i], pl->ev_pool[i], pl->ev_pool[i + 1]));
        }
    }
    *n = have;
    return 0;
}

// ---- NEXT row 1: Heavy State Selection (section 4, Alg. 1) ------------------------------------------------
int tqc_hss_scores(tqc_plan_t *pl, int s, float *scores_dev, void *stream) {
    if (!pl || !scores_dev) return fail(TQC_E_ARG, "null argument");
    const HostPlan &hp = pl->hp;
    if (s < 0 || s >= hp.m) return fail(TQC_E_ARG, "subcircuit id out of range");
    if (!pl->loaded[s]) return fail(TQC_E_STATE, "tensor of subcircuit " + std::to_string(s) + " not loaded");
    if (pl->n_sliced()) return fail(TQC_E_STATE, "state norms need the whole tensor: build the plan without slice_cuts");
    const long long rows = 1ll << hp.o(s);
    const int lgCols = 2 * hp.c(s);
    cudaStream_t st = (cudaStream_t)stream;
    int rc = note_launch(pl, TAG_HSS, st);
    if (rc) return rc;
    const float unscale = std::ldexp(1.0f, hp.d[s]);
    if (rows < 148 * 16 && lgCols >= 10) {                  // few long rows: a block per row keeps every SM loading
        tqc::hss_norm_kernel<256><<<(unsigned)rows, 256, 0, st>>>(pl->d_leaf[s], scores_dev, rows, lgCols, unscale);
    } else {
        const long long warps = std::min<long long>(rows, 148ll * 64 * 32);     // one warp per row: blocks are scheduled as SMs free up
        const unsigned blocks = (unsigned)((warps * 32 + 255) / 256);
        tqc::hss_norm_kernel<32><<<blocks, 256, 0, st>>>(pl->d_leaf[s], scores_dev, rows, lgCols, unscale);
    }
    TQC_CUDA(cudaGetLastError());
    return 0;
}

int tqc_hss_select(const tqc_plan_t *pl, const float *const *scores_host, uint64_t s_max, int32_t *counts, int32_t *keys,
                   size_t keys_capacity) {
    if (!pl || !scores_host || !counts || !keys) return fail(TQC_E_ARG, "null argument");
    const HostPlan &hp = pl->hp;
    struct Cand { float norm; int j, i; };
    std::vector<std::vector<char>> chosen(hp.m);
    std::vector<Cand> rest;
    std::vector<uint64_t> cnt(hp.m, 0);
    size_t total_rows = 0;
    for (int j = 0; j < hp.m; ++j) {
        if (!scores_host[j]) return fail(TQC_E_ARG, "null score array");
        const int n = 1 << hp.o(j);
        total_rows += (size_t)n;
        chosen[j].assign(n, 0);
        for (int i = 0; i < n; ++i)
            if (!std::isfinite(scores_host[j][i])) return fail(TQC_E_ARG, "non-finite score (subcircuit " + std::to_string(j) + ", state " + std::to_string(i) + ")");
        int best = 0;                                       // seed: the heaviest state of every subcircuit (ties: smaller i)
        for (int i = 1; i < n; ++i) if (scores_host[j][i] > scores_host[j][best]) best = i;
        chosen[j][best] = 1; cnt[j] = 1;
        for (int i = 0; i < n; ++i) if (i != best) rest.push_back({scores_host[j][i], j, i});
    }
    if (keys_capacity < total_rows) return fail(TQC_E_ARG, "keys buffer must hold sum_j 2^{o_j} entries");
    // descending norm; ties by smaller subcircuit id, then smaller state (total order: the selection is reproducible)
    std::sort(rest.begin(), rest.end(), [](const Cand &a, const Cand &b) {
        if (a.norm != b.norm) return a.norm > b.norm;
        if (a.j != b.j) return a.j < b.j;
        return a.i < b.i;
    });
    auto product_reached = [&]() {                          // prod_j |x_j| >= s_max, without overflow
        unsigned __int128 p = 1;
        for (int j = 0; j < hp.m; ++j) { p *= cnt[j]; if (p >= s_max) return true; }
        return p >= s_max;
    };
    for (size_t k = 0; k < rest.size() && !product_reached(); ++k) { chosen[rest[k].j][rest[k].i] = 1; cnt[rest[k].j]++; }
    size_t w = 0;
    for (int j = 0; j < hp.m; ++j) {
        counts[j] = (int32_t)cnt[j];
        for (int i = 0; i < (int)chosen[j].size(); ++i) if (chosen[j][i]) keys[w++] = i;      // ascending key order
    }
    return 0;
}

int tqc_hss_expand(const tqc_plan_t *pl, const int32_t *counts, const int32_t *keys, uint64_t *states_host, size_t capacity,
                   size_t *n_states) {
    if (!pl || !counts || !keys || !n_states) return fail(TQC_E_ARG, "null argument");
    const HostPlan &hp = pl->hp;
    unsigned __int128 total = 1;
    for (int j = 0; j < hp.m; ++j) { total *= (uint64_t)std::max(counts[j], 0); if (total > ((unsigned __int128)1 << 40)) return fail(TQC_E_TOO_LARGE, "more than 2^40 composite states"); }
    *n_states = (size_t)total;
    if (!states_host) return 0;
    if (capacity < (size_t)total) return fail(TQC_E_ARG, "states buffer too small");
    const size_t words = (size_t)(hp.n + 63) / 64;
    std::vector<size_t> ofs(hp.m + 1, 0);
    for (int j = 0; j < hp.m; ++j) ofs[j + 1] = ofs[j] + (size_t)counts[j];
    std::vector<int> idx(hp.m, 0);                          // odometer, subcircuit 0 slowest
    for (size_t b = 0; b < (size_t)total; ++b) {
        uint64_t *w = states_host + b * words;
        for (size_t x = 0; x < words; ++x) w[x] = 0;
        for (int j = 0; j < hp.m; ++j) {
            const int key = keys[ofs[j] + idx[j]];
            const int nq = hp.o(j);
            for (int pq = 0; pq < nq; ++pq)                 // first listed qubit = MSB of the key (G4), qubit q = bit q%64 of word q/64 (G5)
                if ((key >> (nq - 1 - pq)) & 1) { const int q = hp.sub_qubits[j][pq]; w[q >> 6] |= 1ull << (q & 63); }
        }
        for (int j = hp.m - 1; j >= 0; --j) { if (++idx[j] < counts[j]) break; idx[j] = 0; }
    }
    return 0;
}

// ---- Heavy State Selection, product-structured contraction ---------------------------------
int tqc_hss_prepare(tqc_plan_t *pl, const int32_t *counts, const int32_t *keys_dev, void *stream) {
    if (!pl || !counts || !keys_dev) return fail(TQC_E_ARG, "null argument");
    const HostPlan &hp = pl->hp;
    if (pl->n_sliced()) return fail(TQC_E_STATE, "pruned contraction needs whole tensors: build the plan without slice_cuts");
    if (hp.m > 64) return fail(TQC_E_TOO_LARGE, "more than 64 subcircuits");
    std::vector<int> v(hp.m, 0);
    int total_bits = 0;
    for (int j = 0; j < hp.m; ++j) {
        if (!pl->loaded[j]) return fail(TQC_E_STATE, "tensor of subcircuit " + std::to_string(j) + " not loaded");
        if (counts[j] < 1 || counts[j] > (1 << hp.o(j))) return fail(TQC_E_ARG, "counts[j] must be in 1 .. 2^{o_j}");
        while ((1 << v[j]) < counts[j]) ++v[j];
        total_bits += v[j];
    }
    if (total_bits > 34) return fail(TQC_E_TOO_LARGE, "padded product of the selections exceeds 2^34 states");
    // same pattern of padded sizes as the last call: keep the plan and its allocations
    bool reuse = pl->hss_sub != nullptr;
    if (reuse) for (int j = 0; j < hp.m; ++j) reuse &= pl->hss_sub->hp.o(j) == v[j];
    if (!reuse) {
        if (pl->hss_sub) { tqc_plan_destroy(pl->hss_sub); pl->hss_sub = nullptr; }
        std::vector<int32_t> cofs(1, 0), cflat, qofs(1, 0), qflat;
        int next_q = 0;                                    // subcircuit 0 owns the most significant virtual bits
        for (int j = 0; j < hp.m; ++j) {
            for (int e : hp.sub_cuts[j]) cflat.push_back(e);
            cofs.push_back((int32_t)cflat.size());
            for (int b = 0; b < v[j]; ++b) qflat.push_back(next_q++);
            qofs.push_back((int32_t)qflat.size());
        }
        std::vector<int32_t> up(hp.cut_up.begin(), hp.cut_up.end()), down(hp.cut_down.begin(), hp.cut_down.end());
        tqc_network_desc d;
        d.n_qubits = total_bits; d.m = hp.m; d.K = hp.K;
        d.cut_up = up.data(); d.cut_down = down.data(); d.sub_cut_ofs = cofs.data(); d.sub_cuts = cflat.data();
        d.sub_qubit_ofs = qofs.data(); d.sub_qubits = qflat.data();
        tqc_plan_opts o;
        memset(&o, 0, sizeof(o));
        o.mode = TQC_MODE_DISTRIBUTION;
        o.use_tcgen05 = pl->use_tcgen05;
        const int rc = tqc_plan(&d, &o, &pl->hss_sub);
        if (rc) { pl->hss_sub = nullptr; return rc; }
    }
    tqc_plan_t *sub = pl->hss_sub;
    cudaStream_t st = (cudaStream_t)stream;
    size_t kofs = 0;
    for (int j = 0; j < hp.m; ++j) {
        const int c = hp.c(j);
        const size_t floats = (size_t)1 << (2 * c + v[j]);
        if (!sub->d_leaf[j]) TQC_CUDA(cudaMalloc(&sub->d_leaf[j], floats * sizeof(float)));
        // digit x of the pruned plan's leaf layout (most significant first) <- the same cut's digit in this plan's layout
        std::vector<int> la = hp.nodes[j].layout, lp = sub->hp.nodes[j].layout;
        if (la.empty()) la = hp.nodes[j].open;
        if (lp.empty()) lp = sub->hp.nodes[j].open;
        BitPairs bp;
        for (int x = 0; x < c; ++x) bp.add_run(2 * (c - 1 - x), 2 * (c - 1 - index_of(la, lp[x])), 2);
        BitMap perm;
        memset(&perm, 0, sizeof(perm));
        if (!bp.build(perm)) return fail(TQC_E_TOO_LARGE, "bit map needs too many segments");
        pl->launches++;
        tqc::hss_rows_kernel<<<(unsigned)std::min<size_t>((floats + 255) / 256, 148 * 32), 256, 0, st>>>(
            pl->d_leaf[j], sub->d_leaf[j], keys_dev + kofs, counts[j], 1ll << v[j], 2 * c, perm);
        TQC_CUDA(cudaGetLastError());
        sub->loaded[j] = 1;
        kofs += (size_t)counts[j];
    }
    pl->hss_counts.assign(counts, counts + hp.m);
    return tqc_plan_finalize(sub, stream);
}

double tqc_hss_cost_log2(const tqc_plan_t *pl) {
    return (pl && pl->hss_sub) ? tqc::cost_log2(pl->hss_sub->hp) : -1.0;
}

size_t tqc_hss_workspace_bytes(const tqc_plan_t *pl) {
    if (!pl || !pl->hss_sub) return 0;
    return align256(((size_t)4) << pl->hss_sub->hp.n) + tqc_plan_workspace_bytes(pl->hss_sub, 0, 0);
}

int tqc_hss_contract(tqc_plan_t *pl, float *out_dev, void *workspace_dev, size_t workspace_bytes, void *stream) {
    if (!pl || !out_dev) return fail(TQC_E_ARG, "null argument");
    if (!pl->hss_sub) return fail(TQC_E_STATE, "call tqc_hss_prepare first");
    if (!workspace_dev || ((uintptr_t)workspace_dev & 255) != 0) return fail(TQC_E_ARG, "workspace must be non-null and 256-byte aligned");
    if (workspace_bytes < tqc_hss_workspace_bytes(pl)) return fail(TQC_E_WORKSPACE, "workspace smaller than tqc_hss_workspace_bytes");
    tqc_plan_t *sub = pl->hss_sub;
    const size_t pb = align256(((size_t)4) << sub->hp.n);
    float *padded = (float *)workspace_dev;
    const uint64_t before = sub->launches;
    int rc = contract_distribution_impl(sub, 0, 0, padded, (char *)workspace_dev + pb, workspace_bytes - pb, stream);
    pl->launches += sub->launches - before;
    if (rc) return rc;
    tqc::HssCompactArgs a;
    memset(&a, 0, sizeof(a));
    a.m = sub->hp.m;
    long long n = 1;
    int shift = 0;
    for (int j = a.m - 1; j >= 0; --j) {                   // subcircuit 0 owns the most significant bits
        a.count[j] = pl->hss_counts[j];
        a.shift[j] = (uint8_t)shift;
        shift += sub->hp.o(j);
        n *= pl->hss_counts[j];
    }
    pl->launches++;
    tqc::hss_compact_kernel<<<(unsigned)std::min<long long>((n + 255) / 256, 148 * 32), 256, 0, (cudaStream_t)stream>>>(padded, out_dev, n, a);
    TQC_CUDA(cudaGetLastError());
    return 0;
}

uint64_t tqc_plan_launch_count(const tqc_plan_t *pl) { return pl ? pl->launches : 0; }
uint64_t tqc_plan_pair_launch_count(const tqc_plan_t *pl) { return pl ? pl->pair_launches : 0; }

int tqc_plan_chain_status(const tqc_plan_t *pl, char *note, size_t note_len) {
    if (!pl) return fail(TQC_E_ARG, "null plan");
    if (note && note_len) { snprintf(note, note_len, "%s", pl->jit_note.c_str()); }
    return !pl->chain ? 0 : (pl->jit_fn ? 2 : 1);
}

// ---- NEXT row 4: subcircuit variants simulated on the device -> T_s (section 2.1) ----------
namespace {
typedef std::pair<double, double> cplx;
// Standard gate definitions written out entry by entry (row-major, first operand = more significant index bit).
bool sim_gate_matrix(int kind, double t, tqc::SimGate &g) {
    const double r = std::sqrt(0.5);
    std::vector<cplx> m;
    auto rot = [&](cplx px00, cplx px01, cplx px10, cplx px11) {       // cos(t/2) I - i sin(t/2) P
        const double c = std::cos(t / 2.0), s = std::sin(t / 2.0);
        auto mi = [&](cplx p) { return cplx(s * p.second, -s * p.first); };   // -i s p
        cplx a = mi(px00), b = mi(px01), cc = mi(px10), d = mi(px11);
        m = {cplx(c + a.first, a.second), b, cc, cplx(c + d.first, d.second)};
    };
    switch (kind) {
    case TQC_GATE_H: m = {{r, 0}, {r, 0}, {r, 0}, {-r, 0}}; break;
    case TQC_GATE_X: m = {{0, 0}, {1, 0}, {1, 0}, {0, 0}}; break;
    case TQC_GATE_Y: m = {{0, 0}, {0, -1}, {0, 1}, {0, 0}}; break;
    case TQC_GATE_Z: m = {{1, 0}, {0, 0}, {0, 0}, {-1, 0}}; break;
    case TQC_GATE_T: m = {{1, 0}, {0, 0}, {0, 0}, {r, r}}; break;             // e^{i pi/4}
    case TQC_GATE_TDG: m = {{1, 0}, {0, 0}, {0, 0}, {r, -r}}; break;
    case TQC_GATE_S: m = {{1, 0}, {0, 0}, {0, 0}, {0, 1}}; break;
    case TQC_GATE_SDG: m = {{1, 0}, {0, 0}, {0, 0}, {0, -1}}; break;
    // exp(-i pi/4 P) = (I - iP)/sqrt2 for P = X, Y, W = (X + Y)/sqrt2 (reading G11)
    case TQC_GATE_SX: m = {{r, 0}, {0, -r}, {0, -r}, {r, 0}}; break;
    case TQC_GATE_SY: m = {{r, 0}, {-r, 0}, {r, 0}, {r, 0}}; break;
    case TQC_GATE_SW: m = {{r, 0}, {-0.5, -0.5}, {0.5, -0.5}, {r, 0}}; break;
    case TQC_GATE_RX: rot({0, 0}, {1, 0}, {1, 0}, {0, 0}); break;
    case TQC_GATE_RY: rot({0, 0}, {0, -1}, {0, 1}, {0, 0}); break;
    case TQC_GATE_RZ: rot({1, 0}, {0, 0}, {0, 0}, {-1, 0}); break;
    case TQC_GATE_CZ:
        m.assign(16, cplx(0, 0));
        m[0] = m[5] = m[10] = cplx(1, 0); m[15] = cplx(-1, 0);
        break;
    case TQC_GATE_CX:                                                   // control = first operand
        m.assign(16, cplx(0, 0));
        m[0] = m[5] = m[11] = m[14] = cplx(1, 0);
        break;
    case TQC_GATE_CP:                                                   // controlled phase: |11> picks up e^{it}
        m.assign(16, cplx(0, 0));
        m[0] = m[5] = m[10] = cplx(1, 0); m[15] = cplx(std::cos(t), std::sin(t));
        break;
    case TQC_GATE_RZZ: {                                                // exp(-i t Z(x)Z): diag e^{-it}, e^{it}, e^{it}, e^{-it}
        m.assign(16, cplx(0, 0));
        const double c = std::cos(t), s = std::sin(t);
        m[0] = m[15] = cplx(c, -s); m[5] = m[10] = cplx(c, s);
        break;
    }
    default: return false;
    }
    g.nq = m.size() == 4 ? 1 : 2;
    for (size_t i = 0; i < m.size(); ++i) g.m[i] = make_double2(m[i].first, m[i].second);
    return true;
}
size_t sim_align(size_t b) { return (b + 255) & ~size_t(255); }

double2 sim_cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// c = a * b for dim x dim row-major complex matrices
void sim_matmul(const double2 *a, const double2 *b, double2 *c, int dim) {
    double2 t[16];
    for (int r = 0; r < dim; ++r)
        for (int col = 0; col < dim; ++col) {
            double2 acc = make_double2(0.0, 0.0);
            for (int k = 0; k < dim; ++k) {
                const double2 p = sim_cmul(a[r * dim + k], b[k * dim + col]);
                acc.x += p.x; acc.y += p.y;
            }
            t[r * dim + col] = acc;
        }
    std::copy(t, t + dim * dim, c);
}
// 4x4 of a one-qubit matrix acting on the first (slot 0) or second (slot 1) operand of a two-qubit op
void sim_lift(const double2 *m, int slot, double2 *out) {
    for (int r = 0; r < 4; ++r)
        for (int c = 0; c < 4; ++c) {
            const int r0 = r >> 1, r1 = r & 1, c0 = c >> 1, c1 = c & 1;
            const bool same = slot == 0 ? r1 == c1 : r0 == c0;
            out[r * 4 + c] = same ? (slot == 0 ? m[r0 * 2 + c0] : m[r1 * 2 + c1]) : make_double2(0.0, 0.0);
        }
}
// Gate fusion (host, exact up to fp64 rounding): every pass over the amplitudes costs the same shared-memory traffic
// whatever the gate, so one-qubit gates are multiplied into the two-qubit op that precedes them on their wire (nothing
// between the two touches that wire), or, before the wire's first two-qubit gate, into the one that follows.  What is
// left is one pass per two-qubit gate plus one per wire that has only one-qubit gates.
std::vector<tqc::SimGate> sim_fuse(const std::vector<tqc::SimGate> &in, int n_in, int w) {
    std::vector<tqc::SimGate> ops;
    std::vector<int> last(w, -1);
    std::vector<char> has_pend(w, 0);
    std::vector<tqc::SimGate> pend(w);
    for (int t = 0; t < n_in; ++t) {
        const tqc::SimGate &g = in[t];
        if (g.nq == 1) {
            const int q = g.b0;
            if (last[q] >= 0) {
                tqc::SimGate &op = ops[last[q]];
                double2 lifted[16];
                sim_lift(g.m, op.b0 == q ? 0 : 1, lifted);
                sim_matmul(lifted, op.m, op.m, 4);
            } else if (has_pend[q]) {
                sim_matmul(g.m, pend[q].m, pend[q].m, 2);
            } else {
                pend[q] = g;
                has_pend[q] = 1;
            }
        } else {
            tqc::SimGate op = g;
            const int qs[2] = {g.b0, g.b1};
            for (int slot = 0; slot < 2; ++slot)
                if (has_pend[qs[slot]]) {
                    double2 lifted[16];
                    sim_lift(pend[qs[slot]].m, slot, lifted);
                    sim_matmul(op.m, lifted, op.m, 4);
                    has_pend[qs[slot]] = 0;
                }
            last[g.b0] = last[g.b1] = (int)ops.size();
            ops.push_back(op);
        }
    }
    for (int q = 0; q < w; ++q)
        if (has_pend[q]) ops.push_back(pend[q]);
    return ops;
}
}  // namespace

namespace {
// grid of sim_variant_kernel: 4^d preparations x 3^g setting groups, g = the smallest split that gives every SM two blocks
// (integers only); w >= 14 keeps at most 2 * 148 blocks so that the per-block amplitudes in the workspace stay L2-resident
void sim_grid(const tqc_subcircuit_desc *sub, unsigned *blocks, int *g_fixed) {
    unsigned b = 1;
    for (int i = 0; i < sub->d && b < (1u << 30); ++i) b *= 4;
    int g = 0;
    while (g < sub->u && b < 2 * 148) { b *= 3; ++g; }
    if (sub->walk_settings == 0 && sub->w <= 13) { for (; g < sub->u && b < (1u << 30); ++g) b *= 3; }     // one block per variant
    *blocks = b; *g_fixed = g;
}
size_t sim_scratch_bytes(const tqc_subcircuit_desc *sub) {
    if (sub->w <= 13) return 0;
    unsigned blocks; int g;
    sim_grid(sub, &blocks, &g);
    return sim_align((size_t)blocks * ((size_t)24 << sub->w));
}
}  // namespace

size_t tqc_simulate_workspace_bytes(const tqc_subcircuit_desc *sub) {
    if (!sub || sub->d < 0 || sub->u < 0 || sub->o < 0 || sub->n_gates < 0 || sub->w < 0 || sub->w > 15 || sub->d > 15 || sub->u > 15) return 0;
    const int lg = 2 * (sub->d + sub->u) + sub->o;
    if (lg > 31) return 0;
    return sim_align(sizeof(tqc::SimGate) * (size_t)std::max(sub->n_gates, 1)) + sim_align(sizeof(double) << lg) + sim_scratch_bytes(sub);
}

int tqc_simulate_subcircuit_tensor(const tqc_subcircuit_desc *sub, float *out_dev, void *workspace_dev,
                                   size_t workspace_bytes, void *stream) {
    if (!sub || !out_dev || !workspace_dev) return fail(TQC_E_ARG, "null argument");
    const int w = sub->w, d = sub->d, u = sub->u, o = sub->o, c = d + u;
    if (w < 0 || d < 0 || u < 0 || o < 0 || sub->n_gates < 0) return fail(TQC_E_ARG, "negative size");
    if (u + o != w) return fail(TQC_E_ARG, "every wire ends in an upstream cut or an output: u + o must equal w");
    if (d > w) return fail(TQC_E_ARG, "more downstream wires than wires");
    if (w > 15) return fail(TQC_E_TOO_LARGE, "w > 15 wires (the paper's subcircuit cap, PAPER.md lines 12-14)");
    if (d > 15 || u > 15 || 2 * c + o > 31) return fail(TQC_E_TOO_LARGE, "4^c 2^o exceeds 2^31 entries");
    if ((d && !sub->D_wires) || (u && !sub->U_wires) || (o && !sub->O_wires) || (c && !sub->bond_pos) ||
        (sub->n_gates && !sub->gates))
        return fail(TQC_E_ARG, "null wire / gate list");
    if ((uintptr_t)workspace_dev & 255) return fail(TQC_E_ARG, "workspace must be 256-byte aligned");
    if (workspace_bytes < tqc_simulate_workspace_bytes(sub)) return fail(TQC_E_WORKSPACE, "workspace too small");
    tqc::SimArgs a{};
    a.w = w; a.d = d; a.u = u; a.o = o; a.n_gates = sub->n_gates;
    std::vector<char> ends(w, 0), begins(w, 0);
    auto wire_ok = [&](int q) { return q >= 0 && q < w; };
    for (int i = 0; i < d; ++i) {
        if (!wire_ok(sub->D_wires[i]) || begins[sub->D_wires[i]]++) return fail(TQC_E_ARG, "bad downstream wire list");
        a.D_bit[i] = w - 1 - sub->D_wires[i];                             // wire 0 = most significant index bit (G4)
    }
    for (int j = 0; j < u; ++j) {
        if (!wire_ok(sub->U_wires[j]) || ends[sub->U_wires[j]]++) return fail(TQC_E_ARG, "bad upstream wire list");
        a.U_bit[j] = w - 1 - sub->U_wires[j];
    }
    for (int j = 0; j < o; ++j) {
        if (!wire_ok(sub->O_wires[j]) || ends[sub->O_wires[j]]++) return fail(TQC_E_ARG, "bad output wire list");
        a.O_bit[j] = w - 1 - sub->O_wires[j];
    }
    tqc::SimPermArgs pa{};
    pa.c = c; pa.o = o;
    std::vector<char> seen(c, 0);
    for (int j = 0; j < c; ++j) {
        const int p = sub->bond_pos[j];
        if (p < 0 || p >= c || seen[p]++) return fail(TQC_E_ARG, "bond_pos is not a permutation of 0..c-1");
        pa.pos[j] = p;
    }
    std::vector<tqc::SimGate> hg((size_t)std::max(sub->n_gates, 1));
    for (int t = 0; t < sub->n_gates; ++t) {
        const tqc_gate &g = sub->gates[t];
        if (!sim_gate_matrix(g.kind, g.param, hg[t])) return fail(TQC_E_ARG, "unknown gate kind " + std::to_string(g.kind));
        if (!wire_ok(g.wire0) || (hg[t].nq == 2 && (!wire_ok(g.wire1) || g.wire1 == g.wire0)))
            return fail(TQC_E_ARG, "gate " + std::to_string(t) + ": wire out of range");
        hg[t].b0 = w - 1 - g.wire0;
        hg[t].b1 = hg[t].nq == 2 ? w - 1 - g.wire1 : 0;
        hg[t].pad = 0;
    }
    const size_t gate_bytes = sim_align(sizeof(tqc::SimGate) * hg.size());     // the workspace is sized for the unfused list
    if (sub->fuse_gates) {
        hg = sim_fuse(hg, sub->n_gates, w);
        a.n_gates = (int)hg.size();
        if (hg.empty()) hg.resize(1);
    }
    cudaStream_t st = (cudaStream_t)stream;
    tqc::SimGate *d_gates = (tqc::SimGate *)workspace_dev;
    a.gates = d_gates;
    a.R = (double *)((char *)workspace_dev + gate_bytes);
    a.scratch = (double2 *)((char *)a.R + sim_align(sizeof(double) << (2 * c + o)));
    // pageable source: the runtime stages the bytes before the call returns, so hg may go out of scope
    TQC_CUDA(cudaMemcpyAsync(d_gates, hg.data(), sizeof(tqc::SimGate) * hg.size(), cudaMemcpyHostToDevice, st));
    const size_t smem = (sizeof(double2) + sizeof(double)) << w;          // amplitudes + probabilities
    { const int arc = ensure_device_attrs(nullptr); if (arc) return arc; }
    // One block per (preparation, group of settings): the settings of the first g upstream wires come from the block id,
    // the block walks the other 3^{u-g}.  g = the smallest split that gives every SM two blocks (integers only).
    unsigned blocks_v = 1;
    int g_fixed = 0;
    sim_grid(sub, &blocks_v, &g_fixed);
    a.g = g_fixed;
    if (w <= 13) {
        // 124 registers per thread: two 256-thread blocks share an SM (the other issues while one waits at a barrier); when
        // the grid cannot give every SM two blocks, one wider block per SM
        tqc::sim_variant_kernel<false><<<blocks_v, (w >= 11 && blocks_v < 2 * 148) ? 512 : 256, smem, st>>>(a);
    } else {
        tqc::sim_variant_kernel<true><<<blocks_v, 512, 0, st>>>(a);        // amplitudes in the workspace (L2), 14-15 wires
    }
    TQC_CUDA(cudaGetLastError());
    const size_t total = size_t(1) << (2 * c + o);
    for (int i = 0; i < d; ++i) {
        const size_t inner = size_t(1) << (2 * (d - 1 - i) + 2 * u + o), tuples = total >> 2;
        const unsigned blocks = (unsigned)std::min<size_t>((tuples + 255) / 256, 148 * 16);
        tqc::sim_kappa_axis_kernel<<<blocks, 256, 0, st>>>(a.R, inner, tuples);
    }
    const unsigned blocks = (unsigned)std::min<size_t>((total + 255) / 256, 148 * 16);
    tqc::sim_permute_cast_kernel<<<blocks, 256, 0, st>>>(a.R, out_dev, pa, total);
    TQC_CUDA(cudaGetLastError());
    return 0;
}

// ---- allocation-free variant of tqc_simulate_subcircuit_tensor (tqc.h: "Callers that cannot allocate") ---------------------
// The gate list and the fp64 result array R of sim_variant_kernel live in ONE file-scope device array instead of a caller's
// workspace.  In host code `tqc_static_scratch` is only the host-side stand-in of the symbol: its device address is looked
// up once per device, with that device current, and that pointer is what the kernels get.
namespace {
static __device__ __align__(256) unsigned char tqc_static_scratch[TQC_STATIC_SCRATCH_BYTES];

int static_scratch_ptr(void **out) {
    static std::mutex mu;
    static void *ptrs[TQC_MAX_DEVICES] = {};
    int dev = 0;
    TQC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= TQC_MAX_DEVICES) return fail(TQC_E_TOO_LARGE, "device ordinal beyond the library's table");
    std::lock_guard<std::mutex> lock(mu);
    if (!ptrs[dev]) {
        void *p = nullptr;
        TQC_CUDA(cudaGetSymbolAddress(&p, tqc_static_scratch));      // the address on the CURRENT device
        if (!p || ((uintptr_t)p & 255)) return fail(TQC_E_CUDA, "static scratch array has no usable device address");
        ptrs[dev] = p;
    }
    *out = ptrs[dev];
    return 0;
}
}  // namespace

size_t tqc_static_scratch_bytes(void) { return (size_t)TQC_STATIC_SCRATCH_BYTES; }

int tqc_simulate_subcircuit_tensor_static(const tqc_subcircuit_desc *sub, float *out_dev, void *stream) {
    if (!sub || !out_dev) return fail(TQC_E_ARG, "null argument");
    const size_t need = tqc_simulate_workspace_bytes(sub);
    if (need == 0) return fail(TQC_E_ARG, "subcircuit description out of range (tqc_simulate_workspace_bytes = 0)");
    if (need > (size_t)TQC_STATIC_SCRATCH_BYTES)
        return fail(TQC_E_TOO_LARGE, "this subcircuit needs " + std::to_string(need) + " bytes of scratch, the static array holds " +
                                         std::to_string((size_t)TQC_STATIC_SCRATCH_BYTES) +
                                         " (tqc_static_scratch_bytes): use tqc_simulate_subcircuit_tensor with a workspace");
    void *scratch = nullptr;
    const int rc = static_scratch_ptr(&scratch);
    if (rc) return rc;
    // the array keeps the last call's contents.  The gate list is overwritten by this call's copy and every entry of R that
    // the later passes read is written by sim_variant_kernel first; R is cleared all the same, so that no value of an
    // earlier call can reach out_dev whatever the description
    const size_t gate_bytes = sim_align(sizeof(tqc::SimGate) * (size_t)std::max(sub->n_gates, 1));
    const size_t r_bytes = sizeof(double) << (2 * (sub->d + sub->u) + sub->o);
    TQC_CUDA(cudaMemsetAsync((char *)scratch + gate_bytes, 0, r_bytes, (cudaStream_t)stream));
    return tqc_simulate_subcircuit_tensor(sub, out_dev, scratch, (size_t)TQC_STATIC_SCRATCH_BYTES, stream);
}

// ---- front half: circuit -> partition -> cuts -> network -> plan (section 6) ----------------------------------------
namespace {
int plan_from_gate_list(int n_qubits, const std::vector<tqc::CircuitGate> &gates, const tqc_cut_opts *cut, const tqc_plan_opts *opts,
                        tqc_plan_t **out) {
    if (!cut || !out) return fail(TQC_E_ARG, "null argument");
    if (n_qubits < 1) return fail(TQC_E_ARG, "n_qubits must be positive");
    if (opts && (opts->n_order_steps > 0 || opts->n_slice_cuts > 0))
        return fail(TQC_E_ARG, "order / slice_cuts name nodes and cuts of a network that does not exist yet: leave them empty");
    tqc::CutOptions co;
    co.w_max = cut->w_max; co.s_max = cut->s_max;
    co.K_t = cut->K_t > 0 ? cut->K_t : 10;
    co.Q_max = cut->Q_max > 0 ? cut->Q_max : 1e4;
    std::string err;
    std::vector<int> part;
    int merges = 0;
    int rc = tqc::greedy_graph_growing(n_qubits, gates, co, part, &merges, err);
    if (rc) return fail(rc, err);
    tqc::CutResult *cr = new tqc::CutResult();
    rc = tqc::extract_subcircuits(n_qubits, gates, part, *cr, err);
    if (rc) { delete cr; return fail(rc, err); }
    cr->merges = merges;
    tqc_network_desc net;
    net.n_qubits = cr->n; net.m = cr->m; net.K = cr->K;
    net.cut_up = cr->cut_up.data(); net.cut_down = cr->cut_down.data();
    net.sub_cut_ofs = cr->sub_cut_ofs.data(); net.sub_cuts = cr->sub_cuts.data();
    net.sub_qubit_ofs = cr->sub_qubit_ofs.data(); net.sub_qubits = cr->sub_qubits.data();
    tqc_plan_t *pl = nullptr;
    rc = tqc_plan(&net, opts, &pl);
    if (rc) { delete cr; return rc; }
    pl->cut = cr;
    *out = pl;
    return 0;
}
}  // namespace

int tqc_plan_from_circuit(const char *circuit_text, const tqc_cut_opts *cut, const tqc_plan_opts *opts, tqc_plan_t **out) {
    int n = 0;
    std::vector<tqc::CircuitGate> gates;
    std::string err;
    const int rc = tqc::parse_circuit_text(circuit_text, n, gates, err);
    if (rc) return fail(rc, err);
    return plan_from_gate_list(n, gates, cut, opts, out);
}

int tqc_plan_from_gates(int n_qubits, const tqc_gate *gates, int n_gates, const tqc_cut_opts *cut, const tqc_plan_opts *opts,
                        tqc_plan_t **out) {
    if (n_gates < 0 || (n_gates > 0 && !gates)) return fail(TQC_E_ARG, "null gate list");
    std::vector<tqc::CircuitGate> gl((size_t)n_gates);
    for (int i = 0; i < n_gates; ++i) {
        const tqc_gate &g = gates[i];
        if (std::string(tqc::gate_name(g.kind)) == "?") return fail(TQC_E_ARG, "gate " + std::to_string(i) + ": unknown kind " + std::to_string(g.kind));
        gl[i].kind = g.kind; gl[i].param = g.param; gl[i].two = tqc::gate_is_two_qubit(g.kind);
        gl[i].q0 = g.wire0; gl[i].q1 = gl[i].two ? g.wire1 : 0;
        if (g.wire0 < 0 || g.wire0 >= n_qubits || (gl[i].two && (g.wire1 < 0 || g.wire1 >= n_qubits || g.wire1 == g.wire0)))
            return fail(TQC_E_ARG, "gate " + std::to_string(i) + ": qubit out of range or duplicate operand");
    }
    return plan_from_gate_list(n_qubits, gl, cut, opts, out);
}

int tqc_plan_cut_network(const tqc_plan_t *pl, tqc_network_desc *net) {
    if (!pl || !net) return fail(TQC_E_ARG, "null argument");
    if (!pl->cut) return fail(TQC_E_STATE, "plan was not made from a circuit");
    const tqc::CutResult &cr = *pl->cut;
    net->n_qubits = cr.n; net->m = cr.m; net->K = cr.K;
    net->cut_up = cr.cut_up.data(); net->cut_down = cr.cut_down.data();
    net->sub_cut_ofs = cr.sub_cut_ofs.data(); net->sub_cuts = cr.sub_cuts.data();
    net->sub_qubit_ofs = cr.sub_qubit_ofs.data(); net->sub_qubits = cr.sub_qubits.data();
    return 0;
}

int tqc_plan_cut_subcircuit(const tqc_plan_t *pl, int s, tqc_subcircuit_desc *sub, int32_t *n2q, int32_t *depth) {
    if (!pl || !sub) return fail(TQC_E_ARG, "null argument");
    if (!pl->cut) return fail(TQC_E_STATE, "plan was not made from a circuit");
    if (s < 0 || s >= pl->cut->m) return fail(TQC_E_ARG, "subcircuit id out of range");
    const tqc::SubcircuitOut &so = pl->cut->subs[s];
    memset(sub, 0, sizeof(*sub));
    sub->w = so.w; sub->n_gates = (int32_t)so.gates.size(); sub->gates = so.gates.data();
    sub->d = (int32_t)so.D_wires.size(); sub->u = (int32_t)so.U_wires.size(); sub->o = (int32_t)so.O_wires.size();
    sub->fuse_gates = 1; sub->walk_settings = 1;
    sub->D_wires = so.D_wires.data(); sub->U_wires = so.U_wires.data(); sub->O_wires = so.O_wires.data();
    sub->bond_pos = so.bond_pos.data();
    if (n2q) *n2q = so.n2q;
    if (depth) *depth = so.depth;
    return 0;
}

int tqc_plan_cut_assignment(const tqc_plan_t *pl, int32_t *part_of_gate, size_t n_gates) {
    if (!pl || (!part_of_gate && n_gates)) return fail(TQC_E_ARG, "null argument");
    if (!pl->cut) return fail(TQC_E_STATE, "plan was not made from a circuit");
    if (n_gates != pl->cut->part_of_gate.size()) return fail(TQC_E_ARG, "n_gates must be " + std::to_string(pl->cut->part_of_gate.size()));
    std::copy(pl->cut->part_of_gate.begin(), pl->cut->part_of_gate.end(), part_of_gate);
    return 0;
}

double tqc_cut_merging_cost(int w_trial, int w_max, int s_trial, int s_max, int K_trial, int K_t) {
    if (w_max < 1 || s_max < 1 || K_t < 1) return -1.0;
    return tqc::merging_cost(w_trial, w_max, s_trial, s_max, K_trial, K_t);
}

// ---- hybrid cost model (section 5, Eqs. 4-6) --------------------------------------------------------------------
int tqc_plan_cost_report(const tqc_plan_t *pl, const tqc_cost_model *model, const int32_t *depth, double n_states, tqc_cost_report *out) {
    if (!pl || !model || !out) return fail(TQC_E_ARG, "null argument");
    if (!(model->flops > 0)) return fail(TQC_E_ARG, "model.flops (floating point operations per second of the classical backend) must be given");
    if (!depth && !pl->cut) return fail(TQC_E_ARG, "depth is needed for a plan that was not made from a circuit");
    const double t_g = model->t_g > 0 ? model->t_g : 1e-7, t_m = model->t_m > 0 ? model->t_m : 1e-6;
    const int n_qpus = model->n_qpus > 0 ? model->n_qpus : 10;
    const int lo = model->shots_log2_min > 0 ? model->shots_log2_min : 10, hi = model->shots_log2_max > 0 ? model->shots_log2_max : 20;
    if (lo > hi) return fail(TQC_E_ARG, "shots_log2_min > shots_log2_max");
    const HostPlan &hp = pl->hp;
    std::vector<int> dn(hp.m, 0), up(hp.m, 0);                      // over the caller's network, sliced cuts included
    for (int s = 0; s < hp.m; ++s) dn[s] = hp.d[s] + (pl->n_sliced() ? pl->d_extra[s] : 0);
    for (int s = 0; s < hp.m; ++s) up[s] = (pl->n_sliced() ? pl->c_full[s] : hp.c(s)) - dn[s];
    double t_qpu = 0, variants = 0;
    for (int s = 0; s < hp.m; ++s) {
        const int w = up[s] + hp.o(s);                               // every wire ends at an upstream cut or at an output
        const int t_i = depth ? depth[s] : pl->cut->subs[s].depth;
        if (t_i < 0) return fail(TQC_E_ARG, "negative depth");
        const double v = std::pow(3.0, up[s]) * std::pow(4.0, dn[s]);
        const double shots = std::ldexp(1.0, std::min(std::max(w, lo), hi));
        variants += v;
        t_qpu += v * shots * ((double)t_i * t_g + t_m);
    }
    t_qpu /= (double)n_qpus;
    double mults = 0;
    for (const Step &st : hp.steps) mults += std::ldexp(1.0, st.log2cost);
    mults *= std::ldexp(1.0, 2 * pl->n_sliced());                    // every sub-network of a sliced plan is contracted
    if (hp.mode == TQC_MODE_STATES) mults *= n_states > 0 ? n_states : 1.0;
    out->c_tn_flop = 2.0 * mults;
    out->t_qpu = t_qpu;
    out->t_classical = out->c_tn_flop / model->flops;
    out->t_total = out->t_qpu + out->t_classical;
    out->qpu_variants = variants;
    return 0;
}

}  // extern "C"
