// Host-side plan: contraction order, node layouts, node kinds, workspace layout.
// Plain C++, no CUDA.  Paper: tensor-network compilation, section 3.5 (lines 441-472);
// cost model of section 3.3 (lines 407-422).  Rules P1-P6 are stated in DESIGN.md.
#pragma once
#include <cstdint>
#include <iterator>
#include <map>
#include <string>
#include <vector>

namespace tqc {

// How a node's tensor is held on the device.
//   LEAF   the re-laid-out subcircuit tensor: 2^{o_s} rows (one per packed key x_s) of 4^{c_s} floats
//   TABLE  an internal node evaluated for EVERY key of its output qubits (rows = 2^{bits}); always in
//          distribution mode, and in states mode while the node carries fewer bits than the batch has
//          states (the per-state values would only repeat)
//   BATCH  an internal node evaluated once per state of the current chunk (rows = states)
enum NodeKind { NODE_LEAF = 0, NODE_TABLE = 1, NODE_BATCH = 2 };

struct Node {
    std::vector<int> open;     // open cut ids, ascending
    std::vector<int> qubits;   // output qubits carried, MSB first (leaf: listed order; inner: lhs || rhs)
    int consumer = -1;         // step that consumes this node (-1: root)
    // device digit layout, most significant first: outer cuts (ascending) then inner cuts
    // (ascending) of the consuming step; root: empty
    std::vector<int> layout;
    int n_inner = 0;           // trailing digits of `layout` that are contracted by the consumer
    int kind = NODE_LEAF;
    int64_t ws_offset = -1;    // BATCH: per-state float offset of this node's block
    int64_t table_offset = -1; // states-mode TABLE: float offset inside the table region
    int key_slot = -1;         // states mode: index of this node's key array (LEAF/TABLE consumed by a BATCH step)
};

struct Step {
    int lhs = 0, rhs = 0;
    std::vector<int> inner, outer_lhs, outer_rhs;   // ascending cut ids
    int log2cost = 0;
    int kernel_class = 0;
};

struct HostPlan {
    int mode = 0, n = 0, m = 0, K = 0, kmax = 0;
    std::vector<int> cut_up, cut_down;
    std::vector<std::vector<int>> sub_cuts;     // caller axis order
    std::vector<std::vector<int>> sub_qubits;
    std::vector<int> d;                         // downstream ends per subcircuit
    std::vector<Node> nodes;                    // m leaves + one per step
    std::vector<Step> steps;
    int64_t ws_floats_per_state = 0;            // states mode: BATCH intermediates, with block reuse
    int64_t table_floats = 0;                   // states mode: TABLE region
    int n_key_slots = 0;
    int table_bits_max = 0, table_log2_floats_max = 0;

    int c(int s) const { return (int)sub_cuts[s].size(); }
    int o(int s) const { return (int)sub_qubits[s].size(); }
    int root() const { return 2 * m - 2; }
};

// first-fit allocator over float offsets, with coalescing free list
struct BlockAlloc {
    std::map<int64_t, int64_t> free_;   // offset -> size
    int64_t top = 0;
    int64_t alloc(int64_t size) {
        for (auto it = free_.begin(); it != free_.end(); ++it) {
            if (it->second >= size) {
                int64_t off = it->first, rem = it->second - size;
                free_.erase(it);
                if (rem > 0) free_[off + size] = rem;
                return off;
            }
        }
        if (!free_.empty()) {   // extend the last free block if it touches the top
            auto last = std::prev(free_.end());
            if (last->first + last->second == top) {
                int64_t off = last->first;
                free_.erase(last);
                top = off + size;
                return off;
            }
        }
        int64_t off = top;
        top += size;
        return off;
    }
    void release(int64_t off, int64_t size) {
        if (size <= 0) return;
        auto it = free_.emplace(off, size).first;
        auto nx = std::next(it);
        if (nx != free_.end() && it->first + it->second == nx->first) {
            it->second += nx->second;
            free_.erase(nx);
        }
        if (it != free_.begin()) {
            auto pv = std::prev(it);
            if (pv->first + pv->second == it->first) {
                pv->second += it->second;
                free_.erase(it);
            }
        }
    }
};

struct PlanOptions {
    int mode = 0;
    std::vector<std::pair<int, int>> order;     // explicit order (empty: greedy)
    int restarts = 0;
    uint64_t seed = 0;
    int kmax_cap = 0;                           // restarts only: prefer orders with K_max <= cap (0: no cap)
    int64_t batch_hint = 0;                     // expected states per call (0: 2^20); sets table_bits_max
    int table_log2_floats_max = 0;              // 0: default 24 (64 MB per table)
    int objective = 0;                          // restarts only: 0 = multiplication count, 1 = modelled run time (states mode)
};

// Structural checks of a network description (ids in range, every cut listed by exactly its two subcircuits, every qubit
// owned once).  Returns 0 or a negative tqc_status; fills err.
int validate_network(int n, int m, int K, const int32_t *cut_up, const int32_t *cut_down, const int32_t *sub_cut_ofs,
                     const int32_t *sub_cuts, const int32_t *sub_qubit_ofs, const int32_t *sub_qubits, std::string &err);

// Returns 0 or a negative tqc_status; fills err.
int build_plan(int n, int m, int K, const int32_t *cut_up, const int32_t *cut_down,
               const int32_t *sub_cut_ofs, const int32_t *sub_cuts, const int32_t *sub_qubit_ofs,
               const int32_t *sub_qubits, const PlanOptions &opts, HostPlan &out, std::string &err);

// modelled run time of the plan's order, femtoseconds per state (states mode; the objective of `objective = 1`)
int64_t plan_time_fs(const HostPlan &p, const PlanOptions &opts);
std::vector<int32_t> serialize_words(const HostPlan &p);
double cost_log2(const HostPlan &p);

// Distribution mode: table sizes depend on the prefix.  free_bits[v] = carried qubits of node v
// with id >= prefix_bits; offsets[v] = float offset of the node's table in the workspace
// (-1 for leaves and for the root, which is written to out[]).  Returns total floats.
int64_t distribution_layout(const HostPlan &p, int prefix_bits, std::vector<int> &free_bits,
                            std::vector<int64_t> &offsets);

}  // namespace tqc
