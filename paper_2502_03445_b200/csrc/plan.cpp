// Host-side planner (plain C++).  See plan.hpp.
//
// P1 leaves are subcircuits 0..m-1; the node created at step t has id m+t.
// P2 candidates: unordered pairs of live nodes sharing >= 1 cut; if none (disconnected
//    network) the pair of the two smallest live ids (outer product).
// P3 two exact integers per candidate: the cost exponent e(a,b) = 2*|E_a u E_b| (PAPER.md lines
//    407-412: a step costs 4^{#inner + #outer}); + o_a + o_b in distribution mode (open output
//    bits carried); and the memory score sigma = size(result) - size(a) - size(b) with
//    size(v) = 2^{w_v} 4^{|E_v|} (w_v = carried output bits in distribution mode, 0 otherwise) --
//    the greedy objective of the order-search library the paper used (CoTenGra, line 449).
// P4 min sigma; tie -> smaller e; tie -> smaller min id; tie -> smaller max id.
// P5 lhs = smaller id; all shared cuts contracted together as one merged bond
//    (PAPER.md lines 318-319), digits ascending by cut id.
// P6 K_max = max_t |E_a u E_b|.
#include "plan.hpp"

#include <algorithm>
#include <cmath>
#include <map>
#include <set>

namespace tqc {

namespace {

constexpr int E_ARG = -1, E_TOO_LARGE = -6;

std::vector<int> set_and(const std::vector<int> &a, const std::vector<int> &b) {
    std::vector<int> r;
    std::set_intersection(a.begin(), a.end(), b.begin(), b.end(), std::back_inserter(r));
    return r;
}
std::vector<int> set_minus(const std::vector<int> &a, const std::vector<int> &b) {
    std::vector<int> r;
    std::set_difference(a.begin(), a.end(), b.begin(), b.end(), std::back_inserter(r));
    return r;
}
std::vector<int> set_xor(const std::vector<int> &a, const std::vector<int> &b) {
    std::vector<int> r;
    std::set_symmetric_difference(a.begin(), a.end(), b.begin(), b.end(), std::back_inserter(r));
    return r;
}
int count_and(const std::vector<int> &a, const std::vector<int> &b) {
    int n = 0;
    size_t i = 0, j = 0;
    while (i < a.size() && j < b.size()) {
        if (a[i] < b[j]) ++i;
        else if (a[i] > b[j]) ++j;
        else { ++n; ++i; ++j; }
    }
    return n;
}

struct SplitMix64 {   // counter-based generator for the randomised restarts (seeded, deterministic)
    uint64_t s;
    explicit SplitMix64(uint64_t seed) : s(seed) {}
    uint64_t next() {
        uint64_t z = (s += 0x9E3779B97F4A7C15ull);
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        return z ^ (z >> 31);
    }
    double uniform() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }
};

// One greedy pass.  noise == 0 -> the deterministic rules P2-P4.  noise > 0 -> the cost
// exponent of each candidate is perturbed by noise * Gumbel-ish jitter (restarts only).
std::vector<std::pair<int, int>> greedy_order(const HostPlan &p, const std::vector<std::vector<int>> &leaf_open,
                                              double noise, SplitMix64 *rng, bool *too_large) {
    const int m = p.m;
    std::map<int, std::vector<int>> open;
    std::map<int, int> obits;
    for (int s = 0; s < m; ++s) { open[s] = leaf_open[s]; obits[s] = p.o(s); }
    std::vector<std::pair<int, int>> order;
    int t = 0;
    while (open.size() > 1) {
        bool have = false;
        double best_score = 0;
        __int128 best_sigma = 0;
        int best_e = 0, best_a = 0, best_b = 0;
        for (auto ia = open.begin(); ia != open.end(); ++ia) {
            auto ib = ia;
            for (++ib; ib != open.end(); ++ib) {
                const int shared = count_and(ia->second, ib->second);
                if (shared == 0) continue;
                const int uni = (int)ia->second.size() + (int)ib->second.size() - shared;
                int e = 2 * uni;
                if (p.mode == 1) e += obits[ia->first] + obits[ib->first];
                const int rest = uni - shared;
                const int wa = p.mode == 1 ? obits[ia->first] : 0, wb = p.mode == 1 ? obits[ib->first] : 0;
                const int xa = wa + 2 * (int)ia->second.size(), xb = wb + 2 * (int)ib->second.size();
                const int xr = wa + wb + 2 * rest;
                if (xr > 120 || xa > 120 || xb > 120) { *too_large = true; return {}; }
                const __int128 sigma = ((__int128)1 << xr) - ((__int128)1 << xa) - ((__int128)1 << xb);
                double score = 0;
                if (noise > 0) {
                    // randomised restarts: jitter the (signed) log of sigma
                    const double mag = std::log2(std::fabs((double)sigma) + 1.0);
                    score = (sigma < 0 ? -mag : mag) +
                            noise * (-std::log(-std::log(rng->uniform() * 0.999998 + 1e-6)));
                }
                bool better;
                if (!have) better = true;
                else if (noise > 0) better = score < best_score;
                else if (sigma != best_sigma) better = sigma < best_sigma;
                else if (e != best_e) better = e < best_e;
                else if (ia->first != best_a) better = ia->first < best_a;
                else better = ib->first < best_b;
                if (better) {
                    have = true;
                    best_score = score; best_sigma = sigma; best_e = e;
                    best_a = ia->first; best_b = ib->first;
                }
            }
        }
        int a, b;
        if (have) { a = best_a; b = best_b; }
        else { auto it = open.begin(); a = it->first; ++it; b = it->first; }
        order.emplace_back(a, b);
        std::vector<int> merged = set_xor(open[a], open[b]);
        int ob = obits[a] + obits[b];
        open.erase(a); open.erase(b); obits.erase(a); obits.erase(b);
        open[m + t] = merged;
        obits[m + t] = ob;
        ++t;
    }
    return order;
}

double order_cost_log2(const HostPlan &p, const std::vector<std::vector<int>> &leaf_open,
                       const std::vector<std::pair<int, int>> &order, int *kmax_out) {
    std::map<int, std::vector<int>> open;
    std::map<int, int> obits;
    for (int s = 0; s < p.m; ++s) { open[s] = leaf_open[s]; obits[s] = p.o(s); }
    double total = 0;   // in units of 2^0; accumulate via log-sum-exp to avoid overflow
    double maxe = -1;
    std::vector<double> es;
    int kmax = 0, t = 0;
    for (auto &ab : order) {
        const auto &A = open[ab.first];
        const auto &B = open[ab.second];
        const int shared = count_and(A, B);
        const int uni = (int)A.size() + (int)B.size() - shared;
        int e = 2 * uni;
        if (p.mode == 1) e += obits[ab.first] + obits[ab.second];
        es.push_back(e);
        maxe = std::max(maxe, (double)e);
        kmax = std::max(kmax, uni);
        std::vector<int> merged = set_xor(A, B);
        int ob = obits[ab.first] + obits[ab.second];
        open.erase(ab.first); open.erase(ab.second);
        open[p.m + t] = merged; obits[p.m + t] = ob;
        ++t;
    }
    for (double e : es) total += std::exp2(e - maxe);
    if (kmax_out) *kmax_out = kmax;
    return es.empty() ? 0.0 : maxe + std::log2(total);
}

// Modelled run time of an order in states mode, femtoseconds per state (integers only, so the choice is reproducible).
// Rates measured on a B200 in round 2 (profiles/r02_tc2_kernel.md, profiles/peaks_r02.md), per fp32-equivalent flop
// (2 per multiplication of PAPER.md lines 407-412):
//   CTA-pair tensor-pipe kernel (both outer dimensions >= 256, K >= 16)   235 TFLOP/s  ->  4.26 fs / flop
//   one-CTA tensor-pipe kernels (larger side >= 128, smaller >= 16, K >= 32)  70 TFLOP/s with a 64-wide narrow side, 20 with a
//                                                                          16-wide one  ->  14 / 50 fs / flop; their per-state
//                                                                          operands stream at 2.4 TB/s (415 fs / byte)
//   fp32 FFMA tile kernel                                                  25 TFLOP/s  ->  40 fs / flop
// plus the bytes of a per-state result that goes through HBM (0.65 / 3.9 TB/s = 167 fs / byte: the stores of a tile overlap
// its successor's MMAs only in part) and of per-state operands read back (200 fs / byte).  A node that carries few output
// bits is a table, evaluated once per key: its cost is spread over the expected batch.
int64_t order_time_fs(const HostPlan &p, const std::vector<std::vector<int>> &leaf_open,
                      const std::vector<std::pair<int, int>> &order, const PlanOptions &opts) {
    const int m = p.m;
    int64_t hint = opts.batch_hint > 0 ? opts.batch_hint : ((int64_t)1 << 20);
    int lg = 0;
    while (((int64_t)2 << lg) <= hint) ++lg;
    const int table_bits_max = std::max(0, lg - 2);
    const int table_log2_floats_max = opts.table_log2_floats_max > 0 ? opts.table_log2_floats_max : 24;
    std::map<int, std::vector<int>> open;
    std::map<int, int> bits, kind;                                  // kind: 0 leaf, 1 table, 2 batch
    for (int s = 0; s < m; ++s) { open[s] = leaf_open[s]; bits[s] = p.o(s); kind[s] = 0; }
    __int128 total = 0;
    int t = 0;
    for (const auto &ab : order) {
        const std::vector<int> &A = open[ab.first], &B = open[ab.second];
        const int shared = count_and(A, B);
        const int lgK = 2 * shared, lgM = 2 * ((int)A.size() - shared), lgN = 2 * ((int)B.size() - shared);
        const int cbits = bits[ab.first] + bits[ab.second], copen = (int)A.size() + (int)B.size() - 2 * shared;
        const bool kids = kind[ab.first] != 2 && kind[ab.second] != 2;
        const bool table = kids && cbits <= table_bits_max && cbits + 2 * copen <= table_log2_floats_max;
        const int e = std::min(lgM + lgN + lgK + 1, 100);            // log2 flops of one row
        __int128 fs;
        if (table) {
            fs = (((__int128)40 << e) << cbits) / hint;              // FFMA / warp-MMA tables, once per key
        } else {
            int fs_per_flop_x100, fs_per_operand_byte = 200;
            const int hi = std::max(lgM, lgN), lo = std::min(lgM, lgN);
            if (lo >= 8 && lgK >= 4) fs_per_flop_x100 = 426;                                   // CTA pairs
            else if (hi >= 7 && lo >= 4 && lgK >= 5) {                                         // one-CTA tensor kernels: the narrow
                fs_per_flop_x100 = lo >= 6 ? 1400 : 5000;                                      // side sets the tile (70 / 20 TFLOP/s)
                fs_per_operand_byte = 415;                                                     // and they stream operands at 2.4 TB/s
            } else fs_per_flop_x100 = 4000;
            fs = ((__int128)fs_per_flop_x100 << e) / 100;
            __int128 rd = 0;
            if (kind[ab.first] == 2) rd += (__int128)fs_per_operand_byte * 4 << std::min(2 * (int)A.size(), 100);
            if (kind[ab.second] == 2) rd += (__int128)fs_per_operand_byte * 4 << std::min(2 * (int)B.size(), 100);
            if (fs_per_operand_byte == 415) fs = std::max(fs, rd);   // narrow tiles: MMAs and the operand stream overlap, the slower one counts
            else fs += rd;
            fs += (__int128)167 * 4 << std::min(2 * copen, 100);     // result bytes
        }
        total += fs;
        std::vector<int> merged = set_xor(A, B);
        open.erase(ab.first); open.erase(ab.second);
        bits.erase(ab.first); bits.erase(ab.second);
        open[m + t] = merged; bits[m + t] = cbits; kind[m + t] = table ? 1 : 2;
        ++t;
    }
    const __int128 cap = ((__int128)1 << 62);
    return (int64_t)std::min(total, cap);
}

// Local search on the contraction TREE (the "subtree reconfiguration" of the order-search library the paper used, PAPER.md
// line 449): a move rewrites X = (P . Q) . Z into (P . Z) . Q or (Q . Z) . P at a random internal node, i.e. it changes which
// pair under X is contracted first; every order is reachable by such rotations.  Simulated annealing on the objective of the
// restarts (multiplication count or modelled run time), seeded, integers and one deterministic generator: the same seed
// gives the same plan.  Returns the best order seen (never worse than the input).
std::vector<std::pair<int, int>> improve_by_rotations(const HostPlan &p, const std::vector<std::vector<int>> &leaf_open,
                                                      std::vector<std::pair<int, int>> order, const PlanOptions &opts,
                                                      int iters, SplitMix64 &rng, int kmax_cap) {
    const int m = p.m, n_nodes = 2 * m - 1;
    if (m < 4 || iters <= 0) return order;
    std::vector<int> left(n_nodes, -1), right(n_nodes, -1), parent(n_nodes, -1);
    for (int t = 0; t < m - 1; ++t) {
        left[m + t] = order[t].first; right[m + t] = order[t].second;
        parent[order[t].first] = m + t; parent[order[t].second] = m + t;
    }
    const int root = n_nodes - 1;
    const bool by_time = opts.objective == 1 && p.mode == 0;
    auto emit = [&](std::vector<std::pair<int, int>> &out) {          // post-order renumbering: children before parents
        out.clear();
        std::vector<int> id(n_nodes, -1), stack = {root}, state(n_nodes, 0);
        for (int s = 0; s < m; ++s) id[s] = s;
        int next = m;
        while (!stack.empty()) {
            const int v = stack.back();
            if (v < m) { stack.pop_back(); continue; }
            if (state[v] == 0) { state[v] = 1; stack.push_back(right[v]); stack.push_back(left[v]); }
            else {
                stack.pop_back();
                if (id[v] >= 0) continue;
                id[v] = next++;
                const int a = id[left[v]], b = id[right[v]];
                out.emplace_back(std::min(a, b), std::max(a, b));
            }
        }
    };
    auto score = [&](const std::vector<std::pair<int, int>> &o, int *kmax) -> double {
        const double c = order_cost_log2(p, leaf_open, o, kmax);
        return by_time ? (double)order_time_fs(p, leaf_open, o, opts) : c;
    };
    std::vector<std::pair<int, int>> cur, best = order, cand;
    emit(cur);
    int k = 0;
    double cur_s = score(cur, &k), best_s = cur_s;
    std::vector<int> internal;
    for (int it = 0; it < iters; ++it) {
        // X: internal node with at least one internal child
        const int X = m + (int)(rng.next() % (uint64_t)(m - 1));
        const bool take_left = (rng.next() & 1) != 0;
        int Y = take_left ? left[X] : right[X], Z = take_left ? right[X] : left[X];
        if (Y < m) { std::swap(Y, Z); if (Y < m) continue; }
        const bool keep_p = (rng.next() & 1) != 0;
        const int P = left[Y], Q = right[Y];
        // new Y = (keep_p ? Q : P) . Z ; new X = Y . (keep_p ? P : Q)
        const int stay = keep_p ? P : Q, join = keep_p ? Q : P;
        left[Y] = join; right[Y] = Z; parent[Z] = Y;
        left[X] = Y; right[X] = stay; parent[stay] = X;
        emit(cand);
        int kc = 0;
        const double s2 = score(cand, &kc);
        const double temp = 0.02 * (double)(iters - it) / (double)iters;             // relative uphill tolerance, cooling to 0
        const double u = rng.uniform();
        const bool cap_ok = kmax_cap <= 0 || kc <= kmax_cap || kc <= k;
        const double cur_cmp = by_time ? cur_s * (1.0 + temp * u) : cur_s + temp * 10.0 * u;
        if (cap_ok && s2 <= cur_cmp) {
            cur_s = s2; k = kc; cur.swap(cand);
            if (s2 < best_s) { best_s = s2; best = cur; }
        } else {                                                                     // undo
            left[Y] = P; right[Y] = Q; parent[Z] = X; parent[stay] = Y;
            if (take_left) { left[X] = Y; right[X] = Z; } else { left[X] = Z; right[X] = Y; }
        }
    }
    return best;
}

}  // namespace

int validate_network(int n, int m, int K, const int32_t *cut_up, const int32_t *cut_down, const int32_t *sub_cut_ofs,
                     const int32_t *sub_cuts, const int32_t *sub_qubit_ofs, const int32_t *sub_qubits, std::string &err) {
    if (n < 0 || m < 1 || K < 0) { err = "n_qubits >= 0, m >= 1, K >= 0 required"; return E_ARG; }
    if (!sub_cut_ofs || !sub_qubit_ofs || (K > 0 && (!cut_up || !cut_down || !sub_cuts)) || (n > 0 && !sub_qubits)) {
        err = "null array in network description"; return E_ARG;
    }
    for (int e = 0; e < K; ++e) {
        if (cut_up[e] < 0 || cut_up[e] >= m || cut_down[e] < 0 || cut_down[e] >= m || cut_up[e] == cut_down[e]) {
            err = "cut " + std::to_string(e) + ": ends must be two distinct subcircuits"; return E_ARG;
        }
    }
    std::vector<int> seen_cut(K, 0), seen_q(n, 0);
    for (int s = 0; s < m; ++s) {
        if (sub_cut_ofs[s + 1] < sub_cut_ofs[s] || sub_qubit_ofs[s + 1] < sub_qubit_ofs[s]) { err = "offsets must ascend"; return E_ARG; }
        std::vector<int> mine;
        for (int j = sub_cut_ofs[s]; j < sub_cut_ofs[s + 1]; ++j) {
            const int e = sub_cuts[j];
            if (e < 0 || e >= K || (cut_up[e] != s && cut_down[e] != s)) {
                err = "subcircuit " + std::to_string(s) + " lists cut " + std::to_string(e) + " it does not touch"; return E_ARG;
            }
            if (std::find(mine.begin(), mine.end(), e) != mine.end()) { err = "duplicate cut in subcircuit"; return E_ARG; }
            mine.push_back(e);
            seen_cut[e]++;
        }
        for (int j = sub_qubit_ofs[s]; j < sub_qubit_ofs[s + 1]; ++j) {
            const int q = sub_qubits[j];
            if (q < 0 || q >= n || seen_q[q]) { err = "output qubit " + std::to_string(q) + " out of range or listed twice"; return E_ARG; }
            seen_q[q] = 1;
        }
        if (sub_qubit_ofs[s + 1] - sub_qubit_ofs[s] > 30) { err = "subcircuit with more than 30 output qubits"; return E_TOO_LARGE; }
    }
    for (int e = 0; e < K; ++e) if (seen_cut[e] != 2) { err = "cut " + std::to_string(e) + " must be listed by exactly its two subcircuits"; return E_ARG; }
    for (int q = 0; q < n; ++q) if (!seen_q[q]) { err = "qubit " + std::to_string(q) + " is owned by no subcircuit"; return E_ARG; }
    return 0;
}

int build_plan(int n, int m, int K, const int32_t *cut_up, const int32_t *cut_down,
               const int32_t *sub_cut_ofs, const int32_t *sub_cuts, const int32_t *sub_qubit_ofs,
               const int32_t *sub_qubits, const PlanOptions &opts, HostPlan &p, std::string &err) {
    if (opts.mode != 0 && opts.mode != 1) { err = "mode must be 0 (states) or 1 (distribution)"; return E_ARG; }
    if (const int vrc = validate_network(n, m, K, cut_up, cut_down, sub_cut_ofs, sub_cuts, sub_qubit_ofs, sub_qubits, err)) return vrc;
    p = HostPlan();
    p.mode = opts.mode; p.n = n; p.m = m; p.K = K;
    p.cut_up.assign(cut_up, cut_up + K);
    p.cut_down.assign(cut_down, cut_down + K);
    p.sub_cuts.resize(m); p.sub_qubits.resize(m); p.d.assign(m, 0);
    for (int s = 0; s < m; ++s) {
        for (int j = sub_cut_ofs[s]; j < sub_cut_ofs[s + 1]; ++j) {
            const int e = sub_cuts[j];
            p.sub_cuts[s].push_back(e);
            if (cut_down[e] == s) p.d[s]++;
        }
        for (int j = sub_qubit_ofs[s]; j < sub_qubit_ofs[s + 1]; ++j) p.sub_qubits[s].push_back(sub_qubits[j]);
        if (p.c(s) > 15) { err = "subcircuit with more than 15 incident cuts"; return E_TOO_LARGE; }
    }

    std::vector<std::vector<int>> leaf_open(m);
    for (int s = 0; s < m; ++s) { leaf_open[s] = p.sub_cuts[s]; std::sort(leaf_open[s].begin(), leaf_open[s].end()); }

    // ---- order ----
    std::vector<std::pair<int, int>> order;
    if (!opts.order.empty()) {
        if ((int)opts.order.size() != m - 1) { err = "explicit order must have m-1 steps"; return E_ARG; }
        std::set<int> live;
        for (int s = 0; s < m; ++s) live.insert(s);
        for (int t = 0; t < m - 1; ++t) {
            int a = opts.order[t].first, b = opts.order[t].second;
            if (a == b || !live.count(a) || !live.count(b)) { err = "explicit order: step " + std::to_string(t) + " uses a dead or unknown node"; return E_ARG; }
            live.erase(a); live.erase(b); live.insert(m + t);
            order.emplace_back(std::min(a, b), std::max(a, b));
        }
    } else {
        bool too_large = false;
        order = greedy_order(p, leaf_open, 0.0, nullptr, &too_large);
        if (too_large) { err = "plan would need a tensor of more than 2^120 entries"; return E_TOO_LARGE; }
        if (opts.restarts > 0) {
            // objective: total multiplication count, among the orders whose K_max (the widest step)
            // stays within kmax_cap; while no order meets the cap the smaller K_max wins
            // (objective = 1, states mode: the modelled run time order_time_fs instead of the multiplication count)
            const bool by_time = opts.objective == 1 && p.mode == 0;
            int best_k = 0;
            double best = order_cost_log2(p, leaf_open, order, &best_k);
            if (by_time) best = (double)order_time_fs(p, leaf_open, order, opts);
            const int cap = opts.kmax_cap > 0 ? opts.kmax_cap : 1 << 30;
            SplitMix64 rng(opts.seed);
            for (int r = 0; r < opts.restarts; ++r) {
                const double noise = 0.5 + 2.5 * (double)(r % 8) / 8.0;
                auto cand = greedy_order(p, leaf_open, noise, &rng, &too_large);
                if (too_large) { too_large = false; continue; }
                int k = 0;
                double c = order_cost_log2(p, leaf_open, cand, &k);
                if (by_time) c = (double)order_time_fs(p, leaf_open, cand, opts);      // exact: the value is an integer < 2^53 in practice
                const bool ok = k <= cap, best_ok = best_k <= cap;
                const bool better = (ok && !best_ok) || (ok == best_ok && (ok ? c < best - (by_time ? 0.5 : 1e-12) : (k < best_k || (k == best_k && c < best - (by_time ? 0.5 : 1e-12)))));
                if (better) { best = c; best_k = k; order = cand; }
            }
            // then tree rotations from the best restart (200 moves per restart asked for)
            order = improve_by_rotations(p, leaf_open, order, opts, std::min(opts.restarts, 1 << 16) * 200, rng, opts.kmax_cap);
        }
    }

    // ---- nodes and steps ----
    p.nodes.assign(m + (m - 1), Node());
    for (int s = 0; s < m; ++s) { p.nodes[s].open = leaf_open[s]; p.nodes[s].qubits = p.sub_qubits[s]; }
    p.steps.resize(m - 1);
    p.kmax = 0;
    for (int t = 0; t < m - 1; ++t) {
        Step &st = p.steps[t];
        st.lhs = order[t].first; st.rhs = order[t].second;
        Node &A = p.nodes[st.lhs], &B = p.nodes[st.rhs], &C = p.nodes[m + t];
        st.inner = set_and(A.open, B.open);
        st.outer_lhs = set_minus(A.open, B.open);
        st.outer_rhs = set_minus(B.open, A.open);
        const int uni = (int)(st.inner.size() + st.outer_lhs.size() + st.outer_rhs.size());
        st.log2cost = 2 * uni + (p.mode == 1 ? (int)(A.qubits.size() + B.qubits.size()) : 0);
        p.kmax = std::max(p.kmax, uni);
        C.open = set_xor(A.open, B.open);
        C.qubits = A.qubits;
        C.qubits.insert(C.qubits.end(), B.qubits.begin(), B.qubits.end());
        A.consumer = t; B.consumer = t;
        A.layout = st.outer_lhs; A.layout.insert(A.layout.end(), st.inner.begin(), st.inner.end());
        B.layout = st.outer_rhs; B.layout.insert(B.layout.end(), st.inner.begin(), st.inner.end());
        A.n_inner = B.n_inner = (int)st.inner.size();
    }
    if (m > 1 && !p.nodes[2 * m - 2].open.empty()) { err = "internal: root has open cuts"; return E_ARG; }
    // Outer digits of each operand in the order they have in the RESULT's layout (root first, so the result's layout is
    // final when its operands are ordered): the result index maps i -> C and j -> C are then order-preserving, the lowest
    // digits of one operand are the lowest digits of C, and a tile of the step covers long contiguous runs of C.
    for (int t = m - 2; t >= 0; --t) {
        const Step &st = p.steps[t];
        const Node &C = p.nodes[m + t];
        for (int op : {st.lhs, st.rhs}) {
            Node &X = p.nodes[op];
            const size_t no = X.layout.size() - (size_t)X.n_inner;
            std::stable_sort(X.layout.begin(), X.layout.begin() + (long)no, [&](int a, int b) {
                const auto ia = std::find(C.layout.begin(), C.layout.end(), a), ib = std::find(C.layout.begin(), C.layout.end(), b);
                return ia < ib;
            });
        }
    }

    // ---- node kinds ----
    {
        int64_t hint = opts.batch_hint > 0 ? opts.batch_hint : ((int64_t)1 << 20);
        int lg = 0;
        while (((int64_t)2 << lg) <= hint) ++lg;            // floor(log2(hint))
        p.table_bits_max = std::max(0, lg - 2);
        p.table_log2_floats_max = opts.table_log2_floats_max > 0 ? opts.table_log2_floats_max : 24;
        for (int t = 0; t < m - 1; ++t) {
            Node &C = p.nodes[m + t];
            const Node &A = p.nodes[p.steps[t].lhs], &B = p.nodes[p.steps[t].rhs];
            if (p.mode == 1) { C.kind = NODE_TABLE; continue; }
            const int bits = (int)C.qubits.size();
            const bool kids = A.kind != NODE_BATCH && B.kind != NODE_BATCH;
            const bool small = bits <= p.table_bits_max && bits + 2 * (int)C.open.size() <= p.table_log2_floats_max;
            C.kind = (kids && small) ? NODE_TABLE : NODE_BATCH;
        }
    }

    // ---- states-mode workspace: table region, key slots, per-state offsets of BATCH nodes ----
    if (p.mode == 0) {
        auto align64 = [](int64_t v) { return (v + 63) / 64 * 64; };
        auto table_size = [&](const Node &v) {
            return align64((int64_t)1 << ((int)v.qubits.size() + 2 * (int)v.open.size()));
        };
        BlockAlloc tal;
        for (int t = 0; t < m - 1; ++t) {
            Node &C = p.nodes[m + t];
            if (C.kind != NODE_TABLE) continue;
            C.table_offset = tal.alloc(table_size(C));
            // a table consumed by another TABLE step is dead afterwards; one consumed by a BATCH
            // step must survive every chunk
            for (int op : {p.steps[t].lhs, p.steps[t].rhs})
                if (op >= m && p.nodes[op].kind == NODE_TABLE) tal.release(p.nodes[op].table_offset, table_size(p.nodes[op]));
        }
        p.table_floats = tal.top;
        BlockAlloc al;
        for (int t = 0; t < m - 1; ++t) {
            Node &C = p.nodes[m + t];
            if (C.kind != NODE_BATCH) continue;
            for (int op : {p.steps[t].lhs, p.steps[t].rhs})
                if (p.nodes[op].kind != NODE_BATCH && p.nodes[op].key_slot < 0) p.nodes[op].key_slot = p.n_key_slots++;
            if (2 * C.open.size() > 40) { err = "an intermediate would hold more than 4^20 values per state"; return E_TOO_LARGE; }
            const int64_t sz = (int64_t)1 << (2 * C.open.size());
            if (t == m - 2) C.ws_offset = -1;             // the root is written straight to out[]
            else C.ws_offset = al.alloc(sz);
            for (int op : {p.steps[t].lhs, p.steps[t].rhs})
                if (p.nodes[op].kind == NODE_BATCH) al.release(p.nodes[op].ws_offset, (int64_t)1 << (2 * p.nodes[op].open.size()));
        }
        p.ws_floats_per_state = al.top;
        // the root is a LEAF (m == 1) or a TABLE (tiny n): out[b] is gathered from it by key
        if (p.nodes[p.root()].kind != NODE_BATCH) p.nodes[p.root()].key_slot = p.n_key_slots++;
    }
    return 0;
}

int64_t distribution_layout(const HostPlan &p, int prefix_bits, std::vector<int> &free_bits,
                            std::vector<int64_t> &offsets) {
    const int m = p.m;
    free_bits.assign(p.nodes.size(), 0);
    offsets.assign(p.nodes.size(), -1);
    for (size_t v = 0; v < p.nodes.size(); ++v)
        for (int q : p.nodes[v].qubits) if (q >= prefix_bits) free_bits[v]++;
    auto align64 = [](int64_t v) { return (v + 63) / 64 * 64; };
    auto size_of = [&](int v) { return align64((int64_t)1 << (free_bits[v] + 2 * (int)p.nodes[v].open.size())); };
    BlockAlloc al;
    for (int t = 0; t < m - 1; ++t) {
        const int v = m + t;
        if (t != m - 2) offsets[v] = al.alloc(size_of(v));
        for (int op : {p.steps[t].lhs, p.steps[t].rhs})
            if (op >= m) al.release(offsets[op], size_of(op));
    }
    return al.top;
}

int64_t plan_time_fs(const HostPlan &p, const PlanOptions &opts) {
    std::vector<std::vector<int>> leaf_open(p.m);
    for (int s = 0; s < p.m; ++s) { leaf_open[s] = p.sub_cuts[s]; std::sort(leaf_open[s].begin(), leaf_open[s].end()); }
    std::vector<std::pair<int, int>> order;
    for (const Step &st : p.steps) order.emplace_back(st.lhs, st.rhs);
    return order_time_fs(p, leaf_open, order, opts);
}

std::vector<int32_t> serialize_words(const HostPlan &p) {
    std::vector<int32_t> w = {p.mode, p.n, p.m, p.K};
    for (const Step &s : p.steps) {
        w.push_back(s.lhs); w.push_back(s.rhs);
        w.push_back((int)s.inner.size()); w.push_back((int)s.outer_lhs.size()); w.push_back((int)s.outer_rhs.size());
        w.push_back(s.log2cost);
        for (int e : s.inner) w.push_back(e);
        for (int e : s.outer_lhs) w.push_back(e);
        for (int e : s.outer_rhs) w.push_back(e);
    }
    w.push_back(p.kmax);
    return w;
}

double cost_log2(const HostPlan &p) {
    if (p.steps.empty()) return 0.0;
    double mx = 0;
    for (const Step &s : p.steps) mx = std::max(mx, (double)s.log2cost);
    double tot = 0;
    for (const Step &s : p.steps) tot += std::exp2((double)s.log2cost - mx);
    return mx + std::log2(tot);
}

}  // namespace tqc
