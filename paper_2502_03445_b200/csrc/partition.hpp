// Host-side front half of tqc_plan_from_circuit (plain C++, no CUDA): circuit text -> gate list -> DAG of two-qubit
// gates (section 6.1.1) -> Greedy Graph Growing partition (Alg. 2) with the edge
// merging cost of Alg. 3 / Table 1 (lines 643-675) under the caps w_max, s_max (lines 596-617) -> cut edges with their
// upstream / downstream ends (section 2.1) -> cut network + one executable description per subcircuit.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/tqc.h"

namespace tqc {

struct CircuitGate {
    int kind = 0;            // TQC_GATE_*
    int q0 = 0, q1 = 0;      // circuit qubits (q1 unused for one-qubit gates)
    double param = 0.0;
    bool two = false;
};

struct CutOptions {
    int w_max = 0, s_max = 0;   // caps: wires per subcircuit, two-qubit gates per subcircuit
    int K_t = 10;               // threshold on the contraction edges of a neighbouring pair
    double Q_max = 1e4;         // merging cost cutoff (line 726)
};

struct SubcircuitOut {
    int w = 0, n2q = 0, depth = 0;
    std::vector<tqc_gate> gates;              // local wires
    std::vector<int32_t> D_wires, U_wires, O_wires, bond_pos;
    std::vector<int32_t> D_cuts, U_cuts, O_qubits;
};

struct CutResult {
    int n = 0, m = 0, K = 0;
    std::vector<int32_t> part_of_gate;        // per circuit gate (one-qubit gates: the subcircuit they were attached to)
    std::vector<int32_t> cut_up, cut_down, cut_qubit;
    std::vector<int32_t> sub_cut_ofs, sub_cuts, sub_qubit_ofs, sub_qubits;
    std::vector<SubcircuitOut> subs;
    int merges = 0;                           // Alg. 2 iterations that merged an edge
};

bool gate_is_two_qubit(int kind);
bool gate_has_param(int kind);
const char *gate_name(int kind);

// "qubits <n>" header, then one gate per line: <name>[(<angle>)] <q0> [<q1>]; '#' starts a comment.
// Returns 0 or TQC_E_PARSE with the line number in err.
int parse_circuit_text(const char *text, int &n_qubits, std::vector<CircuitGate> &gates, std::string &err);

// Table 1: sum of the three terms, or a negative value when a quantum cap is broken ("Not allowed").
double merging_cost(int w_trial, int w_max, int s_trial, int s_max, int K_trial, int K_t);

// Alg. 2 / Alg. 3.  part_of_2q[i] = partition of the i-th two-qubit gate (program order), ids renumbered by first
// appearance.  Returns 0, TQC_E_ARG or TQC_E_INFEASIBLE (a single gate breaks the caps).
int greedy_graph_growing(int n_qubits, const std::vector<CircuitGate> &gates, const CutOptions &opts,
                         std::vector<int> &part_of_2q, int *merges, std::string &err);

// Partition of the two-qubit gates -> cuts, network, subcircuits (conventions in partition.cpp).
int extract_subcircuits(int n_qubits, const std::vector<CircuitGate> &gates, const std::vector<int> &part_of_2q,
                        CutResult &out, std::string &err);

}  // namespace tqc
