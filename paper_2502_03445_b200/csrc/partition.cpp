// See partition.hpp.  Conventions of the extraction (the cut network a partition yields is unique up to numbering; this
// numbering is stated so that an independent implementation can be compared with it):
//   * a WIRE of a subcircuit is a maximal run of same-partition two-qubit gates along one circuit qubit (one run = one
//     qubit of the subcircuit the QPU runs); a qubit no two-qubit gate touches is one wire of subcircuit 0;
//   * a one-qubit gate goes with the nearest PRECEDING two-qubit gate on its qubit, else with the first following one
//     (PAPER.md lines 590-593 says "adjacent"; the side is this library's choice);
//   * cut ids: qubits ascending, then along the wire; the earlier run holds the upstream (measured) end, the later one
//     the downstream (initialised) end (lines 183-187); terminals are never cut (line 594);
//   * local wires of a subcircuit: its runs ordered by (qubit, position along the qubit);
//   * the tensor axes of subcircuit s (tqc_network_desc.sub_cuts) are its incident cut ids ascending; its output qubits
//     (sub_qubits) ascend by circuit qubit.
#include "partition.hpp"

#include <algorithm>
#include <array>
#include <cctype>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>

namespace tqc {

namespace {

struct GateInfo { const char *name; int kind; bool two; bool param; };
const GateInfo kGates[] = {
    {"h", TQC_GATE_H, false, false},     {"x", TQC_GATE_X, false, false},     {"s", TQC_GATE_S, false, false},
    {"sdg", TQC_GATE_SDG, false, false}, {"sx", TQC_GATE_SX, false, false},   {"sy", TQC_GATE_SY, false, false},
    {"sw", TQC_GATE_SW, false, false},   {"rx", TQC_GATE_RX, false, true},    {"ry", TQC_GATE_RY, false, true},
    {"rz", TQC_GATE_RZ, false, true},    {"cz", TQC_GATE_CZ, true, false},    {"cx", TQC_GATE_CX, true, false},
    {"rzz", TQC_GATE_RZZ, true, true},   {"y", TQC_GATE_Y, false, false},     {"z", TQC_GATE_Z, false, false},
    {"t", TQC_GATE_T, false, false},     {"tdg", TQC_GATE_TDG, false, false}, {"cp", TQC_GATE_CP, true, true},
};
const GateInfo *info_of(int kind) {
    for (const GateInfo &g : kGates) if (g.kind == kind) return &g;
    return nullptr;
}

}  // namespace

bool gate_is_two_qubit(int kind) { const GateInfo *g = info_of(kind); return g && g->two; }
bool gate_has_param(int kind) { const GateInfo *g = info_of(kind); return g && g->param; }
const char *gate_name(int kind) { const GateInfo *g = info_of(kind); return g ? g->name : "?"; }

int parse_circuit_text(const char *text, int &n_qubits, std::vector<CircuitGate> &gates, std::string &err) {
    n_qubits = -1;
    gates.clear();
    if (!text) { err = "null circuit text"; return TQC_E_PARSE; }
    int line_no = 0;
    const char *p = text;
    while (*p) {
        const char *eol = strchr(p, '\n');
        std::string line(p, eol ? (size_t)(eol - p) : strlen(p));
        p = eol ? eol + 1 : p + line.size();
        ++line_no;
        const size_t hash = line.find('#');
        if (hash != std::string::npos) line.resize(hash);
        // tokens: split on blanks; "(...)" stays attached to the gate name
        std::vector<std::string> tok;
        size_t i = 0;
        while (i < line.size()) {
            while (i < line.size() && isspace((unsigned char)line[i])) ++i;
            if (i >= line.size()) break;
            size_t j = i;
            int depth = 0;
            while (j < line.size() && (depth > 0 || !isspace((unsigned char)line[j]))) {
                if (line[j] == '(') ++depth;
                if (line[j] == ')') --depth;
                ++j;
            }
            tok.push_back(line.substr(i, j - i));
            i = j;
        }
        if (tok.empty()) continue;
        auto fail_line = [&](const std::string &what) { err = "line " + std::to_string(line_no) + ": " + what; return (int)TQC_E_PARSE; };
        auto parse_int = [&](const std::string &s, int &v) {
            if (s.empty()) return false;
            char *end = nullptr;
            const long x = strtol(s.c_str(), &end, 10);
            if (*end != '\0' || x < 0 || x > 1000000) return false;
            v = (int)x;
            return true;
        };
        if (n_qubits < 0) {
            if (tok.size() != 2 || tok[0] != "qubits" || !parse_int(tok[1], n_qubits) || n_qubits < 1) return fail_line("expected the header `qubits <n>`");
            continue;
        }
        std::string name = tok[0], arg;
        const size_t par = name.find('(');
        if (par != std::string::npos) {
            if (name.back() != ')') return fail_line("unbalanced parenthesis");
            arg = name.substr(par + 1, name.size() - par - 2);
            name.resize(par);
        }
        const GateInfo *gi = nullptr;
        for (const GateInfo &g : kGates) if (name == g.name) gi = &g;
        if (!gi) return fail_line("unknown gate `" + name + "`");
        CircuitGate g;
        g.kind = gi->kind; g.two = gi->two;
        if (gi->param) {
            if (arg.empty()) return fail_line("gate `" + name + "` takes one angle");
            char *end = nullptr;
            g.param = strtod(arg.c_str(), &end);
            while (*end && isspace((unsigned char)*end)) ++end;
            if (*end != '\0' || !std::isfinite(g.param)) return fail_line("bad angle `" + arg + "`");
        } else if (par != std::string::npos) return fail_line("gate `" + name + "` takes no parameter");
        if ((int)tok.size() != (gi->two ? 3 : 2)) return fail_line("gate `" + name + "` takes " + (gi->two ? "two operands" : "one operand"));
        if (!parse_int(tok[1], g.q0) || g.q0 >= n_qubits) return fail_line("qubit index out of range");
        if (gi->two) {
            if (!parse_int(tok[2], g.q1) || g.q1 >= n_qubits) return fail_line("qubit index out of range");
            if (g.q1 == g.q0) return fail_line("duplicate operand");
        }
        gates.push_back(g);
    }
    if (n_qubits < 0) { err = "missing `qubits <n>` header"; return TQC_E_PARSE; }
    return 0;
}

double merging_cost(int w_trial, int w_max, int s_trial, int s_max, int K_trial, int K_t) {
    if (w_trial > w_max || s_trial > s_max) return -1.0;                    // quantum hard constraints: "Not allowed"
    double q = (double)w_trial / (double)w_max + (double)s_trial / (double)s_max;
    if (K_trial <= K_t) q += (double)K_trial / (double)K_t;                 // x / T
    else q += (K_trial - K_t > 500 ? HUGE_VAL : std::pow(4.0, (double)(K_trial - K_t))) + 1.0;   // 4^{x-T} + 1
    return q;
}

namespace {
// One partition of the growing graph.  With s two-qubit gates and `internal` same-qubit consecutive gate pairs inside it,
// its wire count is w = 2 s - internal (every gate brings two qubit incidences, every internal pair joins two runs).
struct Part {
    int s = 0, internal = 0, deg = 0;          // deg = cut edges leaving the partition
    std::map<int, int> nb;                     // neighbour id -> crossing wire segments X(a, b)
    bool alive = true;
};
}  // namespace

int greedy_graph_growing(int n_qubits, const std::vector<CircuitGate> &gates, const CutOptions &opts,
                         std::vector<int> &part_of_2q, int *merges, std::string &err) {
    if (opts.w_max < 1 || opts.s_max < 1 || opts.K_t < 1 || !(opts.Q_max > 0)) { err = "w_max, s_max, K_t, Q_max must be positive"; return TQC_E_ARG; }
    std::vector<int> g2;                                        // indices of the two-qubit gates (the DAG's vertices)
    for (size_t i = 0; i < gates.size(); ++i) if (gates[i].two) g2.push_back((int)i);
    const int V = (int)g2.size();
    part_of_2q.assign(V, 0);
    if (merges) *merges = 0;
    if (V == 0) return 0;
    if (opts.w_max < 2) { err = "w_max < 2: a single two-qubit gate already needs two qubits"; return TQC_E_INFEASIBLE; }
    // DAG edges: consecutive two-qubit gates on a qubit wire (terminal segments are never cut)
    std::vector<Part> parts(V);
    std::vector<int> last(n_qubits, -1);
    for (int v = 0; v < V; ++v) {
        parts[v].s = 1;
        const CircuitGate &g = gates[g2[v]];
        for (int q : {g.q0, g.q1}) {
            if (last[q] >= 0) {
                const int u = last[q];
                parts[u].nb[v]++; parts[v].nb[u]++;
                parts[u].deg++; parts[v].deg++;
            }
            last[q] = v;
        }
    }
    std::vector<int> owner(V);
    for (int v = 0; v < V; ++v) owner[v] = v;
    // Alg. 3 for the candidate (a, b): trial-merge, count, un-merge (nothing is modified: the counts are closed forms)
    auto cost_of = [&](int a, int b) -> double {
        const Part &A = parts[a], &B = parts[b];
        const int x = A.nb.at(b);
        const int s_trial = A.s + B.s;
        const int w_trial = (2 * A.s - A.internal) + (2 * B.s - B.internal) - x;
        const int deg_t = A.deg + B.deg - 2 * x;
        int k_trial = 0;                                      // max over the trial partition's neighbours c of K_{T,c}
        auto visit = [&](int c, int xc) { k_trial = std::max(k_trial, deg_t + parts[c].deg - xc); };
        for (const auto &kv : A.nb) {
            if (kv.first == b) continue;
            const auto it = B.nb.find(kv.first);
            visit(kv.first, kv.second + (it == B.nb.end() ? 0 : it->second));
        }
        for (const auto &kv : B.nb) if (kv.first != a && !A.nb.count(kv.first)) visit(kv.first, kv.second);
        return merging_cost(w_trial, opts.w_max, s_trial, opts.s_max, k_trial, opts.K_t);
    };
    for (;;) {
        // every candidate is re-evaluated each round: a merge changes deg() of the new partition, which enters the K term
        // of its neighbours' other candidates too (PAPER.md lines 636-638 update "all neighboring edges")
        int ba = -1, bb = -1;
        double bq = 0;
        for (int a = 0; a < V; ++a) {
            if (!parts[a].alive) continue;
            for (const auto &kv : parts[a].nb) {
                const int b = kv.first;
                if (b <= a) continue;
                const double q = cost_of(a, b);
                if (q < 0 || q > opts.Q_max) continue;
                if (ba < 0 || q < bq) { ba = a; bb = b; bq = q; }    // ties: the pair met first = smaller (a, b)
            }
        }
        if (ba < 0) break;
        Part &A = parts[ba], &B = parts[bb];
        const int x = A.nb.at(bb);
        A.s += B.s;
        A.internal += B.internal + x;
        A.deg = A.deg + B.deg - 2 * x;
        A.nb.erase(bb);
        for (const auto &kv : B.nb) {
            if (kv.first == ba) continue;
            A.nb[kv.first] += kv.second;
            Part &C = parts[kv.first];
            C.nb[ba] += kv.second;
            C.nb.erase(bb);
        }
        B.alive = false; B.nb.clear();
        for (int v = 0; v < V; ++v) if (owner[v] == bb) owner[v] = ba;
        if (merges) ++*merges;
    }
    // renumber by first appearance in program order
    std::map<int, int> id;
    for (int v = 0; v < V; ++v) {
        auto it = id.find(owner[v]);
        if (it == id.end()) it = id.emplace(owner[v], (int)id.size()).first;
        part_of_2q[v] = it->second;
    }
    return 0;
}

int extract_subcircuits(int n_qubits, const std::vector<CircuitGate> &gates, const std::vector<int> &part_of_2q,
                        CutResult &out, std::string &err) {
    out = CutResult();
    out.n = n_qubits;
    const int G = (int)gates.size();
    std::vector<int> idx2(G, -1);
    int V = 0;
    for (int i = 0; i < G; ++i) if (gates[i].two) idx2[i] = V++;
    if ((int)part_of_2q.size() != V) { err = "partition must assign every two-qubit gate"; return TQC_E_ARG; }
    struct Seg { int qubit, idx, part, cut_in, cut_out, local; };
    std::vector<Seg> segs;
    std::vector<std::vector<int>> wire_segs(n_qubits), twoq(n_qubits);
    std::vector<std::array<int, 2>> seg_of(G, std::array<int, 2>{-1, -1});    // per gate operand
    for (int i = 0; i < G; ++i) {
        if (!gates[i].two) continue;
        if (part_of_2q[idx2[i]] < 0) { err = "negative partition id"; return TQC_E_ARG; }
        twoq[gates[i].q0].push_back(i);
        twoq[gates[i].q1].push_back(i);
    }
    for (int q = 0; q < n_qubits; ++q) {
        if (twoq[q].empty()) {
            segs.push_back({q, 0, 0, -1, -1, -1});
            wire_segs[q].push_back((int)segs.size() - 1);
            continue;
        }
        for (int gi : twoq[q]) {
            const int part = part_of_2q[idx2[gi]];
            int sid;
            if (!wire_segs[q].empty() && segs[wire_segs[q].back()].part == part) sid = wire_segs[q].back();
            else {
                segs.push_back({q, (int)wire_segs[q].size(), part, -1, -1, -1});
                sid = (int)segs.size() - 1;
                wire_segs[q].push_back(sid);
            }
            seg_of[gi][gates[gi].q0 == q ? 0 : 1] = sid;
        }
    }
    for (int i = 0; i < G; ++i) {
        if (gates[i].two) continue;
        const int q = gates[i].q0;
        int before = -1;
        for (int gi : twoq[q]) if (gi < i) before = gi;
        if (before >= 0) seg_of[i][0] = seg_of[before][gates[before].q0 == q ? 0 : 1];
        else if (!twoq[q].empty()) { const int f = twoq[q][0]; seg_of[i][0] = seg_of[f][gates[f].q0 == q ? 0 : 1]; }
        else seg_of[i][0] = wire_segs[q][0];
    }
    for (int q = 0; q < n_qubits; ++q)
        for (size_t x = 0; x + 1 < wire_segs[q].size(); ++x) {
            const int a = wire_segs[q][x], b = wire_segs[q][x + 1], e = (int)out.cut_up.size();
            out.cut_up.push_back(segs[a].part); out.cut_down.push_back(segs[b].part); out.cut_qubit.push_back(q);
            segs[a].cut_out = e; segs[b].cut_in = e;
        }
    out.K = (int)out.cut_up.size();
    int m = 0;
    for (const Seg &s : segs) m = std::max(m, s.part + 1);
    out.m = m;
    out.subs.assign(m, SubcircuitOut());
    std::vector<int> order(segs.size());
    for (size_t i = 0; i < segs.size(); ++i) order[i] = (int)i;
    std::sort(order.begin(), order.end(), [&](int a, int b) {
        if (segs[a].part != segs[b].part) return segs[a].part < segs[b].part;
        if (segs[a].qubit != segs[b].qubit) return segs[a].qubit < segs[b].qubit;
        return segs[a].idx < segs[b].idx;
    });
    for (int sid : order) {
        Seg &s = segs[sid];
        SubcircuitOut &sub = out.subs[s.part];
        s.local = sub.w;
        if (s.cut_in >= 0) { sub.D_wires.push_back(sub.w); sub.D_cuts.push_back(s.cut_in); }
        if (s.cut_out >= 0) { sub.U_wires.push_back(sub.w); sub.U_cuts.push_back(s.cut_out); }
        else { sub.O_wires.push_back(sub.w); sub.O_qubits.push_back(s.qubit); }
        sub.w++;
    }
    out.part_of_gate.assign(G, 0);
    std::vector<std::vector<int>> layer(m);
    for (int s = 0; s < m; ++s) layer[s].assign(out.subs[s].w, 0);
    for (int i = 0; i < G; ++i) {
        const int part = segs[seg_of[i][0]].part;
        if (gates[i].two && segs[seg_of[i][1]].part != part) { err = "internal: gate operands in different subcircuits"; return TQC_E_ARG; }
        out.part_of_gate[i] = part;
        SubcircuitOut &sub = out.subs[part];
        tqc_gate g;
        memset(&g, 0, sizeof(g));
        g.kind = gates[i].kind; g.param = gates[i].param;
        g.wire0 = segs[seg_of[i][0]].local;
        g.wire1 = gates[i].two ? segs[seg_of[i][1]].local : 0;
        sub.gates.push_back(g);
        sub.n2q += gates[i].two ? 1 : 0;
        // depth t_i: layers of an as-soon-as-possible schedule of the subcircuit's gates
        int l = layer[part][g.wire0];
        if (gates[i].two) l = std::max(l, layer[part][g.wire1]);
        ++l;
        layer[part][g.wire0] = l;
        if (gates[i].two) layer[part][g.wire1] = l;
        sub.depth = std::max(sub.depth, l);
    }
    out.sub_cut_ofs.assign(1, 0); out.sub_qubit_ofs.assign(1, 0);
    for (int s = 0; s < m; ++s) {
        SubcircuitOut &sub = out.subs[s];
        std::vector<int32_t> mine = sub.D_cuts;
        mine.insert(mine.end(), sub.U_cuts.begin(), sub.U_cuts.end());
        std::vector<int32_t> sorted = mine;
        std::sort(sorted.begin(), sorted.end());
        for (int32_t e : mine) sub.bond_pos.push_back((int32_t)(std::find(sorted.begin(), sorted.end(), e) - sorted.begin()));
        out.sub_cuts.insert(out.sub_cuts.end(), sorted.begin(), sorted.end());
        out.sub_cut_ofs.push_back((int32_t)out.sub_cuts.size());
        out.sub_qubits.insert(out.sub_qubits.end(), sub.O_qubits.begin(), sub.O_qubits.end());
        out.sub_qubit_ofs.push_back((int32_t)out.sub_qubits.size());
    }
    return 0;
}

}  // namespace tqc
