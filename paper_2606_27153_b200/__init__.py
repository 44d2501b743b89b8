"""libdmuon for B200: the single-GPU Muon optimizer step of DMuon (arxiv/paper_2606_27153).

`binding` is the ctypes layer over the C ABI of include/dmuon.h (same names, marshalling only);
`synth` draws the seeded synthetic inputs; `build` compiles libdmuon.so in-tree.
"""
from . import binding, synth  # noqa: F401
from .binding import (DmuonError, adamw_step, adamw_step_noalloc, assign_owners, measure_cost, block_schedule, describe_plan, ns_sym_mm, muon_step, muon_step_host, muon_step_master, ns_batched, ns_batched_sched, ns_gemm, profile_read,  # noqa: F401
                      profile_reset, set_option, set_workspace, shutdown, version, warmup, workspace_bytes)
