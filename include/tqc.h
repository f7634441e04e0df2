/* tqc.h — C ABI of the B200-native TensorQC reconstruction library (libtqc.so).
 *
 * What the library computes (arXiv 2502.03445, "TensorQC"; PAPER.md = /root/reference/PAPER.md):
 *
 *     p(x) = 2^{-K} * sum_{k in {I,X,Y,Z}^K}  prod_{s=1..m}  T_s[ idx_s(k), x_s ]
 *
 * i.e. Eq. 1 with the factor 1/2 per cut the printed equation omits
 * (reading G1), evaluated not as the 4^K-term sum but as a tensor-network
 * contraction of the subcircuit output tensors over their 4-valued cut-edge bonds
 * (section 3.2-3.3): m-1 pairwise contractions, parallel cuts merged
 * into one bond, any order giving the same value (lines 343-348, 397-399).
 *
 * Conventions (readings G4-G6):
 *   - Basis index order I=0, X=1, Y=2, Z=3.
 *   - Subcircuit tensor T_s is [4^{c_s}][2^{o_s}] row-major fp32 (trailing output axis); the
 *     first listed incident cut of s is the most significant base-4 digit of the row index.
 *   - x_s packs the output qubits of s in their listed order, first = MSB.
 *   - A distribution index is i = sum_q x_q 2^{n-1-q} (qubit 0 = MSB).
 *   - A batch state is ceil(n/64) uint64 words; qubit q is bit (q % 64) of word (q / 64).
 *
 * Every call returns 0 on success or a negative tqc_status; tqc_last_error() gives a
 * thread-local message.  No exception crosses the boundary.  Pointers are marked HOST or
 * DEVICE.  The library never synchronises the caller's stream inside the contract calls and
 * never allocates there: persistent device state (re-laid-out tensors) is allocated in
 * tqc_load_subcircuit_tensors; the plan's device tables, the plan-specialised chain kernel (an NVRTC
 * compile) and the side streams of forked table steps are created by tqc_plan_finalize, which the
 * load that completes the tensor set calls; scratch comes from the caller's workspace.  A contract
 * call is therefore capturable in a CUDA graph from the first call on.  (Exception: with
 * tqc_plan_profile_enable on, a contract call creates the CUDA events it records.)
 * A plan is not re-entrant: at most one load / contract call per plan at a time, and consecutive
 * calls on one plan must be ordered on the device (same stream, or the caller's own events);
 * different plans are independent.  Attributes of the library's kernels are set per device.
 * A release build of the library reads no environment variable.
 * There is no CPU fallback: without a CUDA device the compute calls fail with TQC_E_CUDA.
 */
#ifndef TQC_H
#define TQC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    TQC_OK = 0,
    TQC_E_ARG = -1,        /* null pointer, out-of-range id, inconsistent description */
    TQC_E_SHAPE = -2,      /* n_elems does not match 4^{c_s} * 2^{o_s} */
    TQC_E_STATE = -3,      /* a tensor has not been loaded / wrong mode for this call */
    TQC_E_INFEASIBLE = -4, /* partitioning caps cannot be met */
    TQC_E_WORKSPACE = -5,  /* workspace too small (see tqc_plan_workspace_bytes) */
    TQC_E_TOO_LARGE = -6,  /* a dimension exceeds what the library indexes */
    TQC_E_CUDA = -7,       /* CUDA runtime error (message has the CUDA string) */
    TQC_E_PARSE = -8       /* circuit text could not be parsed */
} tqc_status;

enum { TQC_MODE_STATES = 0, TQC_MODE_DISTRIBUTION = 1 };

/* Kernel class chosen per plan step (integer thresholds):
 * SIMT_TILE  register-tiled fp32 FFMA contraction (any shape);
 * DOT        final reduction: no outer cuts left, one dot product over the merged bond per state;
 * TCGEN05    3xTF32 tcgen05.mma / TMEM / TMA contraction for steps with large outer dimensions;
 * CHAIN      the step is part of the fused small-bond chain: all per-state steps of the plan run in one kernel, one
 *            warp per state, intermediates in shared memory, bond sums finished by warp shuffles. */
enum { TQC_KERNEL_SIMT_TILE = 0, TQC_KERNEL_DOT = 1, TQC_KERNEL_TCGEN05 = 2, TQC_KERNEL_CHAIN = 3 };
/* TCGEN05 steps with both outer dimensions >= 256 run step_tc2_kernel: 256 x 256 tiles over CTA pairs (cta_group::2), which
 * halve the operand bytes per flop; the others run the one-CTA kernel step_tc_kernel<BN>. */
/* How a node of the contraction tree is evaluated. */
enum { TQC_NODE_LEAF = 0, TQC_NODE_TABLE = 1, TQC_NODE_BATCH = 2 };

typedef struct tqc_plan tqc_plan_t;

/* Cut network (cut set E, subcircuits C_1..C_m, E_i subset of E).
 * All arrays HOST, caller-owned, copied by tqc_plan. */
typedef struct {
    int32_t n_qubits;               /* n */
    int32_t m;                      /* subcircuits */
    int32_t K;                      /* wire cuts |E| */
    const int32_t *cut_up;          /* [K] subcircuit holding the upstream (measured) end of cut e */
    const int32_t *cut_down;        /* [K] subcircuit holding the downstream (initialised) end */
    const int32_t *sub_cut_ofs;     /* [m+1] offsets into sub_cuts */
    const int32_t *sub_cuts;        /* incident cut ids of s in the AXIS ORDER of the caller's T_s */
    const int32_t *sub_qubit_ofs;   /* [m+1] offsets into sub_qubits */
    const int32_t *sub_qubits;      /* output qubits of s, first = MSB of x_s; every qubit exactly once */
} tqc_network_desc;

typedef struct {
    int32_t mode;                   /* TQC_MODE_STATES or TQC_MODE_DISTRIBUTION */
    int32_t n_order_steps;          /* 0: greedy planner (rules P1-P6); else m-1 explicit steps */
    const int32_t *order;           /* HOST [2*n_order_steps] (lhs, rhs) node ids; leaves 0..m-1, step t creates m+t */
    int32_t restarts;               /* >0: seeded randomised-greedy restarts, best total cost kept (not bit-pinned) */
    uint64_t seed;
    int64_t batch_hint;             /* states mode: expected n_states per call (0 = 2^20).  A node that carries at most
                                       log2(batch_hint) - 2 output bits is evaluated once per KEY (a table) instead of
                                       once per state.  Any n_states is still legal at contract time. */
    int32_t table_log2_floats_max;  /* 0 = default 24: cap on log2(entries) of such a table */
    int32_t use_tcgen05;            /* 0 = default (on where a step qualifies), -1 = never (fp32 FFMA everywhere) */
    int32_t use_chain;              /* 0 = default (fused chain kernel when every per-state step is small, specialised for
                                       the plan at the first contract call), -1 = never, -2 = fused but not specialised */
    int32_t n_slice_cuts;           /* index slicing (Fig. 6): these cut edges are not contracted as   */
    const int32_t *slice_cuts;      /* bonds; the network is evaluated once per assignment of their bases (4^{n_slice_cuts}
                                       smaller networks, planned once) and the results are summed.  HOST [n_slice_cuts] distinct
                                       cut ids.  Tensors are still loaded whole; every intermediate that carried a sliced cut is 4x
                                       smaller per cut.  Sliced plans run step by step (no fused chain); workspace sizes include
                                       one partial-sum buffer (4 bytes per output of a chunk). */
    int32_t kmax_cap;               /* restarts > 0 only: among the randomised-greedy orders keep the cheapest one whose widest
                                       step K_max = max_t |E_a u E_b| is <= kmax_cap; while no order meets the
                                       cap the smaller K_max wins.  0 = no cap (total multiplication count only). */
    int32_t objective;              /* restarts > 0 only: 0 = keep the order with the fewest multiplications; 1 (states mode) = keep
                                       the order with the smallest MODELLED RUN TIME: per step, flops over the measured rate of the
                                       kernel class the step would get (CTA-pair tensor pipe / one-CTA tensor pipe / FFMA) plus the
                                       HBM bytes of per-state results and operands; integers only, deterministic per seed
                                       (csrc/plan.cpp order_time_fs; tqc_plan_modelled_seconds_per_state reports it) */
} tqc_plan_opts;

/* ---- planning (host only; no CUDA call) -------------------------------------------------
 * tqc_plan: network description -> contraction order (section 3.5.1;
 * the paper delegates this to CoTenGra, this library ships a deterministic greedy planner)
 * + device layouts + kernel class per step.  *out is library-owned until tqc_plan_destroy. */
int tqc_plan(const tqc_network_desc *net, const tqc_plan_opts *opts, tqc_plan_t **out);
/* Which cuts to slice: the paper's two-level strategy, host only, deterministic.
 * Level 1 - while a subcircuit tensor of one sub-network (4^{c'_s} 2^{o_s} floats, c'_s = unsliced incident cuts) exceeds
 *   2^{max_log2_input_floats}: slice "the most size-reducing cut edge", i.e. among the cuts touching an oversize tensor
 *   the one whose two tensors are largest (larger one first, then the smaller one; tie: smaller cut id).
 * Level 2 - while the largest intermediate of the greedy plan (4^{open cuts} floats per state, x 2^{carried output bits}
 *   in distribution mode) exceeds 2^{max_log2_intermediate_floats}: slice the cut whose removal leaves the smallest
 *   largest-intermediate, then the smallest total multiplication count, then the smaller id (one plan per candidate).
 * slice_cuts: HOST [K] out, in pick order; *n_slice_cuts out.  opts supplies mode / planner options (order is ignored).
 * TQC_E_INFEASIBLE when a limit cannot be met.  Pass the result as tqc_plan_opts.slice_cuts. */
int tqc_choose_slice_cuts(const tqc_network_desc *net, const tqc_plan_opts *opts, int max_log2_input_floats,
                          int max_log2_intermediate_floats, int32_t *slice_cuts, int32_t *n_slice_cuts);
void tqc_plan_destroy(tqc_plan_t *plan);

int tqc_plan_mode(const tqc_plan_t *plan);
int tqc_plan_num_qubits(const tqc_plan_t *plan);
int tqc_plan_num_subcircuits(const tqc_plan_t *plan);
int tqc_plan_num_cuts(const tqc_plan_t *plan);                   /* K of the caller's network (sliced cuts included) */
int tqc_plan_num_sliced_cuts(const tqc_plan_t *plan);
int tqc_plan_num_steps(const tqc_plan_t *plan);
int tqc_plan_kmax(const tqc_plan_t *plan);                       /* max_t |E_a u E_b| */
int tqc_plan_tensor_shape(const tqc_plan_t *plan, int s, int *c_s, int *o_s);
/* step i: operands, #inner, #outer_lhs, #outer_rhs, log2 of its multiplication count
 * (4^{#inner+#outer}; + open output bits in distribution mode), kernel class */
int tqc_plan_step(const tqc_plan_t *plan, int i, int *lhs, int *rhs, int *n_inner,
                  int *n_outer_lhs, int *n_outer_rhs, int *log2cost, int *kernel_class);
/* node v (leaves 0..m-1, then one per step): kind (TQC_NODE_*), carried output bits, open cuts */
int tqc_plan_node(const tqc_plan_t *plan, int v, int *kind, int *n_bits, int *n_open);
/* log2 of the total multiplication count sum_t 2^{log2cost_t} (per state in states mode) */
double tqc_plan_cost_log2(const tqc_plan_t *plan);
/* the run-time model of tqc_plan_opts.objective = 1 evaluated on this plan (states mode; negative otherwise) */
double tqc_plan_modelled_seconds_per_state(const tqc_plan_t *plan);
/* Serialised plan (little-endian int32 words, format in DESIGN.md "Plan blob"): the object
 * compared byte-for-byte with the reference planner.  Call with buf = NULL to get *len. */
int tqc_plan_serialize(const tqc_plan_t *plan, void *buf /*HOST*/, size_t *len);
/* Workspace bytes that let tqc_contract_states process n_states in ONE chunk (a smaller
 * workspace is legal down to tqc_plan_workspace_min_bytes: the batch is then chunked), or
 * that tqc_contract_distribution needs for the given prefix_bits (pass n_states = 0). */
size_t tqc_plan_workspace_bytes(const tqc_plan_t *plan, size_t n_states, int prefix_bits);
size_t tqc_plan_workspace_min_bytes(const tqc_plan_t *plan);

/* ---- a1: load + re-layout (the subcircuit output as a tensor) ----
 * data: [4^{c_s}][2^{o_s}] row-major fp32, HOST (on_device = 0) or DEVICE (on_device = 1).
 * The library copies it into its own device buffer, state-major [2^{o_s}][4^{c_s}] with the
 * bond digits permuted for the plan and multiplied by the exact 2^{-d_s} (sum_s d_s = K);
 * the caller may free `data` once `stream` has completed.  Reloading replaces the tensor. */
int tqc_load_subcircuit_tensors(tqc_plan_t *plan, int s, const float *data, size_t n_elems,
                                int on_device, void *stream /* cudaStream_t */);

/* Completes a plan whose tensors are all loaded: device copies of the key-slot tables, the fused chain's step table and its
 * plan-specialised kernel (NVRTC; if libnvrtc is missing the generic chain kernel is kept and tqc_plan_chain_status says
 * so), side streams / events, kernel attributes of the current device.  May allocate and synchronise.  Called implicitly by
 * the tqc_load_subcircuit_tensors call that loads the last missing tensor; calling it again is a no-op.  TQC_E_STATE if a
 * tensor is missing.  The contract calls return TQC_E_STATE on a plan that was never finalized. */
int tqc_plan_finalize(tqc_plan_t *plan, void *stream /* cudaStream_t */);

/* ---- a2-a5: states mode ------------------------------------------------------------------
 * out_dev[b] = p(x_b) for b < n_states.  states_dev: DEVICE [n_states][ceil(n/64)] uint64.
 * Asynchronous on `stream`; workspace_dev DEVICE, caller-owned, 256-byte aligned. */
int tqc_contract_states(tqc_plan_t *plan, const uint64_t *states_dev, size_t n_states,
                        float *out_dev, void *workspace_dev, size_t workspace_bytes, void *stream);

/* ---- a6: distribution mode ---------------------------------------------------------------
 * out_dev[i] = p(x) for the 2^{n-prefix_bits} bitstrings whose first prefix_bits qubits equal
 * prefix_value (qubit 0 = MSB of prefix_value's prefix_bits-bit field), i enumerating the
 * remaining qubits, lowest-numbered remaining qubit = MSB.  Plan must be MODE_DISTRIBUTION. */
int tqc_contract_distribution(tqc_plan_t *plan, uint64_t prefix_value, int prefix_bits,
                              float *out_dev, void *workspace_dev, size_t workspace_bytes, void *stream);

/* ---- the same two calls with HOST buffers (end-to-end form; "reconstruct
 * 1 million arbitrary quantum states" handed over by the host program) -----------------------
 * states_host / out_host: HOST (pinned memory makes the copies asynchronous).  The library
 * stages them inside the caller's DEVICE workspace, which must hold
 * tqc_plan_workspace_bytes_host(plan, n_states, prefix_bits) bytes for a single chunk (states
 * mode accepts less, down to staging + tqc_plan_workspace_min_bytes).  Order on `stream`:
 * H2D copy of the states, the contraction kernels, D2H copy of the result; the caller
 * synchronises `stream` before reading out_host. */
size_t tqc_plan_workspace_bytes_host(const tqc_plan_t *plan, size_t n_states, int prefix_bits);
int tqc_contract_states_host(tqc_plan_t *plan, const uint64_t *states_host, size_t n_states,
                             float *out_host, void *workspace_dev, size_t workspace_bytes, void *stream);
int tqc_contract_distribution_host(tqc_plan_t *plan, uint64_t prefix_value, int prefix_bits,
                                   float *out_host, void *workspace_dev, size_t workspace_bytes,
                                   void *stream);

/* ---- Heavy State Selection (section 4, Algorithm 1) -- first row of SURVEY 8(f) -----------------
 * tqc_hss_scores: scores_dev[i] = ||p_{s,i}|| = sqrt(sum_e T_s[e, i]^2) for every binary state i of subcircuit s
 *   (the L2 norm over all edge permutations, Alg. 1 line 3), DEVICE [2^{o_s}], asynchronous on `stream`; the tensor
 *   must be loaded.  Scores refer to the caller's values (the 2^{-d_s} folded in at load is undone exactly).
 * tqc_hss_select (host only): Alg. 1 on the m score arrays (HOST, scores_host[j] has 2^{o_j} entries): every subcircuit
 *   is seeded with its heaviest state (ties: smaller i), the remaining (j, i) are taken in descending norm (ties: smaller
 *   j, then smaller i) while prod_j |x_j| < s_max (readings: seeds count toward the product, the last addition may
 *   overshoot s_max, the loop also ends when everything is selected).  counts[j] = |x_j|; keys = the selected states of
 *   subcircuit 0, then 1, ..., each ascending (HOST, capacity >= sum_j 2^{o_j}).
 * tqc_hss_expand (host only): the prod_j |x_j| composite states in the batch format of tqc_contract_states (G5), product
 *   order with subcircuit 0 slowest.  Call with states_host = NULL to get *n_states. */
int tqc_hss_scores(tqc_plan_t *plan, int s, float *scores_dev, void *stream);
int tqc_hss_select(const tqc_plan_t *plan, const float *const *scores_host, uint64_t s_max, int32_t *counts, int32_t *keys,
                   size_t keys_capacity);
int tqc_hss_expand(const tqc_plan_t *plan, const int32_t *counts, const int32_t *keys, uint64_t *states_host, size_t capacity,
                   size_t *n_states);

/* Product-structured contraction of a selection ("prune subcircuit outputs prior to tensor network
 * contraction", output dimension prod_j |x_j|): every subcircuit tensor is restricted to its selected states and the
 * network is contracted ONCE with those pruned output axes open, so the prod_j |x_j| composite states share every
 * intermediate - the same values as tqc_contract_states on tqc_hss_expand's batch, at a fraction of the work.
 * tqc_hss_prepare (allocates, like a load): counts HOST [m] = |x_j|; keys_dev DEVICE [sum_j counts[j]] = the selected
 *   states of subcircuit 0, then 1, ... (the order of tqc_hss_select's keys).  Builds the pruned tensors on `stream` from
 *   the loaded ones and plans the pruned network (axes padded to powers of two; at most 2^34 padded composite states).
 * tqc_hss_contract: out_dev DEVICE [prod_j counts[j]] in product order, subcircuit 0 slowest (tqc_hss_expand's order);
 *   workspace >= tqc_hss_workspace_bytes(plan), 256-byte aligned; asynchronous on `stream`, no allocation. */
int tqc_hss_prepare(tqc_plan_t *plan, const int32_t *counts, const int32_t *keys_dev, void *stream);
size_t tqc_hss_workspace_bytes(const tqc_plan_t *plan);
/* log2 of the multiplication count of the pruned contraction tqc_hss_prepare planned (all padded composite states
 * together, the count of tqc_plan_cost_log2 in distribution mode); negative before tqc_hss_prepare.  Host only. */
double tqc_hss_cost_log2(const tqc_plan_t *plan);
int tqc_hss_contract(tqc_plan_t *plan, float *out_dev, void *workspace_dev, size_t workspace_bytes, void *stream);

/* ---- Subcircuit variants on the device (section 2.1) -- fourth row of SURVEY 8(f) ---------------
 * The quantum half of the method runs every subcircuit in 4^{d_s} * 3^{u_s} variants - each downstream cut wire
 * initialised in |0>, |1>, |+> or |i>, each upstream cut wire measured in Z, X or Y (I shares the Z setting, lines
 * 184-185) - and the Pauli bases of a downstream cut are "constructed as a linear combination from the initialization
 * states" (line 188; coefficients: DESIGN.md reading G3).  tqc_simulate_subcircuit_tensor stands in for the QPU with a
 * noiseless fp64 statevector simulation of all variants on the device ("noiseless classical simulators", line 722) and
 * writes T_s in the layout tqc_load_subcircuit_tensors takes with on_device = 1.
 *
 * sub (HOST, read before the call returns):
 *   w wires; wire 0 is the most significant bit of the amplitude index (G4); all wires start in |0> unless listed in D.
 *     w = 0 (a subcircuit no gate was assigned to) gives the 1 x 1 tensor [1].
 *   gates[n_gates] applied in order; kind = TQC_GATE_*, wire0 (and wire1 for two-qubit gates; CX controls on wire0),
 *     param = angle of RX/RY/RZ (exp(-i param P / 2)), of RZZ (exp(-i param Z(x)Z): the FULL angle, not param / 2) and of
 *     CP (phase e^{i param} on |11>); SX/SY/SW = exp(-i pi/4 P) for P = X, Y, (X+Y)/sqrt2; T / TDG = diag(1, e^{+-i pi/4}).
 *   D_wires[d]: wires that begin at a downstream cut end;  U_wires[u]: wires that end at an upstream cut end;
 *   O_wires[o]: wires that end at a circuit output, in the order of x_s (first = MSB).  u + o = w.
 *   bond_pos[d + u]: bond j (D_wires in order, then U_wires in order) is digit bond_pos[j] of the row index of T_s
 *     (0 = most significant = the subcircuit's first listed incident cut).
 * out_dev DEVICE [4^{d+u}][2^o] fp32.  workspace DEVICE, 256-byte aligned, >= tqc_simulate_workspace_bytes(sub) (0 if the
 * description is out of range).  Asynchronous on `stream`, no allocation.  Errors: TQC_E_ARG (inconsistent lists, unknown
 * gate), TQC_E_TOO_LARGE (w > 15 or 4^{d+u} 2^o > 2^31), TQC_E_WORKSPACE, TQC_E_CUDA.
 * Up to 13 wires the 2^w complex128 amplitudes of a variant stay in one block's shared memory; 14- and 15-wire subcircuits (the
 * paper's cap) keep them in the workspace, which then also holds 24 * 2^w bytes per thread block. */
enum { TQC_GATE_H = 0, TQC_GATE_X = 1, TQC_GATE_S = 2, TQC_GATE_SDG = 3, TQC_GATE_SX = 4, TQC_GATE_SY = 5, TQC_GATE_SW = 6,
       TQC_GATE_RX = 7, TQC_GATE_RY = 8, TQC_GATE_RZ = 9, TQC_GATE_CZ = 10, TQC_GATE_CX = 11, TQC_GATE_RZZ = 12,
       TQC_GATE_Y = 13, TQC_GATE_Z = 14, TQC_GATE_T = 15, TQC_GATE_TDG = 16,
       TQC_GATE_CP = 17 /* controlled phase diag(1, 1, 1, e^{i param}) */ };
typedef struct {
    int32_t kind, wire0, wire1, reserved;
    double param;
} tqc_gate;
typedef struct {
    int32_t w, n_gates;
    const tqc_gate *gates;
    int32_t d, u, o;
    int32_t fuse_gates; /* 1: one-qubit gates are multiplied into the neighbouring two-qubit gate on their wire (one pass per
                           two-qubit gate; same unitary up to fp64 rounding); 0: one pass per listed gate */
    const int32_t *D_wires, *U_wires, *O_wires, *bond_pos;
    int32_t walk_settings; /* 1: a block simulates a preparation once and walks several measurement settings from that
                              state (Gray-code order, one rotation pass per setting); 0: one block per variant */
    int32_t reserved;
} tqc_subcircuit_desc;
size_t tqc_simulate_workspace_bytes(const tqc_subcircuit_desc *sub);
int tqc_simulate_subcircuit_tensor(const tqc_subcircuit_desc *sub, float *out_dev, void *workspace_dev,
                                   size_t workspace_bytes, void *stream);

/* ---- Callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc) -------------------
 * tqc_simulate_subcircuit_tensor_static is tqc_simulate_subcircuit_tensor (same section of the paper, lines 182-192; same
 * kernels, same results) with NO workspace argument: the scratch of the simulation kernel - the device copy of the gate list
 * and the fp64 array R [4^{d+u}][2^o] the variants are accumulated in - lives in one array of TQC_STATIC_SCRATCH_BYTES (8 MiB)
 * that is part of the library image: every GPU that loads the library holds those 8 MiB until the process exits, and the call
 * itself calls no cudaMalloc, cudaFree or allocating library routine (host side: a std::vector of the gate list).
 *   sub, out_dev, stream: as for tqc_simulate_subcircuit_tensor (sub HOST, out_dev DEVICE [4^{d+u}][2^o] fp32, caller-owned).
 *   Limit: tqc_simulate_workspace_bytes(sub) <= tqc_static_scratch_bytes() = 8 MiB, i.e. w <= 13 wires and roughly
 *   4^{d+u} 2^o <= 2^19 entries with a few thousand gates; anything larger returns TQC_E_TOO_LARGE (the message names both
 *   sizes) and launches nothing - use the workspace entry point for it.  Other errors as tqc_simulate_subcircuit_tensor.
 *   The device must be current when the call is made (the array's address is looked up once per device).
 *   The array is SHARED by every call on a device and keeps the last call's contents: the part a call reads is cleared or
 *   overwritten by that call first, so calls that follow one another on one stream (or are ordered by events) are
 *   independent; two calls that may OVERLAP on the GPU (different streams, different host threads) race on it - order them. */
#define TQC_STATIC_SCRATCH_BYTES (8u << 20)
size_t tqc_static_scratch_bytes(void);
int tqc_simulate_subcircuit_tensor_static(const tqc_subcircuit_desc *sub, float *out_dev, void *stream);

/* ---- Front half: circuit -> DAG -> partition -> cuts -> network -> plan (section 6) ---------------
 * The circuit is cut by partitioning its two-qubit gates (lines 578-594: the DAG keeps only two-qubit gates, a one-qubit
 * gate follows its adjacent two-qubit gate, input / output terminals are never cut) with Greedy Graph Growing (Alg. 2,
 * lines 624-641): starting from one partition per two-qubit gate, repeatedly merge the pair of neighbouring partitions with
 * the smallest merging cost Q_e <= Q_max (ties: the pair with the smaller partition ids), where Alg. 3 / Table 1 (lines
 * 643-675) give Q_e = w_trial / w_max + s_trial / s_max + (K_trial / K_t if K_trial <= K_t else 4^{K_trial - K_t} + 1);
 * w_trial = wires of the merged partition (one per maximal run of its gates along a qubit), s_trial = its two-qubit gates,
 * K_trial = max over its neighbours c of the cut edges a pairwise contraction with c would carry (inner + outer); a merge
 * with w_trial > w_max or s_trial > s_max is not allowed (lines 596-617).  Every wire segment between two partitions is
 * a cut, upstream end in the earlier partition (lines 183-187).  Numbering conventions: csrc/partition.cpp.
 * Deterministic: the same circuit and options give the same partition.
 *
 * tqc_plan_from_circuit: circuit_text HOST, NUL-terminated: "qubits <n>" then one gate per line, <name>[(<angle>)] <q0> [<q1>]
 *   with names h x y z s sdg t tdg sx sy sw rx ry rz cz cx cp rzz, '#' comments.  TQC_E_PARSE names the offending line.
 * tqc_plan_from_gates: the same from a gate list (wire0 / wire1 = circuit qubits).
 * cut: w_max, s_max required (> 0); K_t = 0 -> 10, Q_max = 0 -> 1e4 (line 726).  TQC_E_INFEASIBLE when a single gate breaks
 *   the caps.  opts as for tqc_plan (order / slice_cuts must be empty: the network does not exist yet).
 * The plan owns the cut description; the queries below expose it (pointers stay valid until tqc_plan_destroy):
 *   tqc_plan_cut_network     the tqc_network_desc the plan was built from;
 *   tqc_plan_cut_subcircuit  subcircuit s as a tqc_subcircuit_desc ready for tqc_simulate_subcircuit_tensor (fuse_gates = 1,
 *                            walk_settings = 1), its two-qubit gate count and its depth t_s (ASAP layers, line 531);
 *   tqc_plan_cut_assignment  per gate of the circuit, the subcircuit it went to (HOST [n_gates]). */
typedef struct {
    int32_t w_max, s_max;   /* caps: qubits (wires) and two-qubit gates per subcircuit */
    int32_t K_t;            /* 0 = 10 */
    int32_t reserved;
    double Q_max;           /* 0 = 1e4 */
} tqc_cut_opts;
int tqc_plan_from_circuit(const char *circuit_text, const tqc_cut_opts *cut, const tqc_plan_opts *opts, tqc_plan_t **out);
int tqc_plan_from_gates(int n_qubits, const tqc_gate *gates, int n_gates, const tqc_cut_opts *cut, const tqc_plan_opts *opts,
                        tqc_plan_t **out);
int tqc_plan_cut_network(const tqc_plan_t *plan, tqc_network_desc *net);
int tqc_plan_cut_subcircuit(const tqc_plan_t *plan, int s, tqc_subcircuit_desc *sub, int32_t *n_two_qubit_gates, int32_t *depth);
int tqc_plan_cut_assignment(const tqc_plan_t *plan, int32_t *part_of_gate, size_t n_gates);
/* Table 1 alone (host): the merging cost of a trial partition, or a negative value when a cap is broken ("Not allowed"). */
double tqc_cut_merging_cost(int w_trial, int w_max, int s_trial, int s_max, int K_trial, int K_t);

/* ---- Hybrid cost model (section 5, Eqs. 4-6) -------------------------------------------------------
 * T_QPU = sum_i 3^{u_i} 4^{d_i} shots_i (t_i t_g + t_m) / n_qpus,  shots_i = 2^{w_i} kept within [2^shots_log2_min,
 * 2^shots_log2_max] ("the number of shots equal to the number of quantum states per subcircuit, with limits ranging from
 * 2^10 to 2^20", lines 523-524);  T_classical = C_TN / flops with C_TN = 2 x the plan's multiplication count (x n_states in
 * states mode);  T = T_QPU + T_classical (Eq. 6).  Zero fields take the paper's values: t_g = 1e-7 s, t_m = 1e-6 s (lines
 * 520-521), n_qpus = 10 (line 724), shots limits 10 and 20; flops must be given.  depth HOST [m] = t_i per subcircuit, or
 * NULL for a plan made by tqc_plan_from_circuit / _gates (its own depths; any other plan then fails with TQC_E_ARG). */
typedef struct {
    double t_g, t_m, flops;
    int32_t n_qpus, shots_log2_min, shots_log2_max, reserved;
} tqc_cost_model;
typedef struct {
    double t_qpu, t_classical, t_total;   /* seconds */
    double c_tn_flop;                     /* C_TN */
    double qpu_variants;                  /* sum_i 3^{u_i} 4^{d_i}: subcircuit variants to run */
} tqc_cost_report;
int tqc_plan_cost_report(const tqc_plan_t *plan, const tqc_cost_model *model, const int32_t *depth, double n_states,
                         tqc_cost_report *out);

/* ---- measurement hooks (bench.py) --------------------------------------------------------------
 * tqc_plan_launch_count: kernels launched so far on behalf of this plan.
 * tqc_plan_profile_enable(plan, 1): every later contract call records one CUDA event on the
 * caller's stream before each of its kernel launches and one at its end.
 * tqc_plan_profile_read: waits for the last profiled call and returns, per launch in launch
 * order, its tag (plan step index t >= 0; -1 key extraction; -2 root gather) and the time to the
 * next event in ms.  Call with tags = NULL to get the count in *n.  HOST arrays. */
uint64_t tqc_plan_launch_count(const tqc_plan_t *plan);
/* of those, launches of step_tc2_kernel (tcgen05 cta_group::2 tiles over CTA pairs, csrc/kernels_tc2.cuh) */
uint64_t tqc_plan_pair_launch_count(const tqc_plan_t *plan);
/* 0: the plan does not use the fused chain kernel; 1: it runs the generic (table-driven) chain kernel; 2: it runs the chain
 * kernel specialised for this plan (the library generates the plan's steps as straight-line CUDA from its own templates
 * in csrc/kernels_chain.cuh and compiles them with NVRTC at the first contract call; if NVRTC is not available the
 * generic kernel runs).  note (HOST, may be NULL) receives a one-line explanation. */
int tqc_plan_chain_status(const tqc_plan_t *plan, char *note, size_t note_len);
int tqc_plan_profile_enable(tqc_plan_t *plan, int on);
int tqc_plan_profile_read(tqc_plan_t *plan, int32_t *tags, float *ms, size_t *n);

const char *tqc_last_error(void);
const char *tqc_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TQC_H */
