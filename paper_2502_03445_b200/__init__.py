"""B200-native TensorQC reconstruction hot path (arXiv 2502.03445): thin Python binding over the
C-ABI library libtqc.so (include/tqc.h).  Argument marshalling only; every step of the path runs
in the CUDA kernels under csrc/.  There is no CPU fallback: without the built library the import
of `binding` fails, and without a CUDA device the compute calls return TQC_E_CUDA."""
from .binding import (MODE_DISTRIBUTION, MODE_STATES, Plan, TqcError, lib_path, tqc_contract_distribution,
                      tqc_contract_distribution_host, tqc_contract_states, tqc_contract_states_host,
                      tqc_choose_slice_cuts, tqc_hss_contract, tqc_hss_expand, tqc_hss_scores, tqc_hss_select, tqc_load_subcircuit_tensors, tqc_plan,
                      tqc_simulate_subcircuit_tensor, tqc_simulate_workspace_bytes,
                      tqc_simulate_subcircuit_tensor_static, tqc_static_scratch_bytes,
                      tqc_plan_from_circuit, tqc_plan_from_gates, tqc_cut_merging_cost, circuit_text, version)

__all__ = ["MODE_STATES", "MODE_DISTRIBUTION", "Plan", "TqcError", "tqc_plan", "tqc_load_subcircuit_tensors",
           "tqc_contract_states", "tqc_contract_distribution", "tqc_contract_states_host",
           "tqc_contract_distribution_host", "tqc_hss_scores", "tqc_hss_select", "tqc_hss_expand", "tqc_hss_contract", "tqc_choose_slice_cuts", "tqc_simulate_subcircuit_tensor",
           "tqc_simulate_workspace_bytes", "tqc_simulate_subcircuit_tensor_static", "tqc_static_scratch_bytes", "tqc_plan_from_circuit", "tqc_plan_from_gates", "tqc_cut_merging_cost",
           "circuit_text", "version",
           "lib_path"]
