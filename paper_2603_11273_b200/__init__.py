"""B200-native hot path of duration-aware ASR scheduling (arxiv 2603.11273).

Thin ctypes binding over ``libasr_sched.so`` (``include/asr_sched.h``): every
function here only marshals arguments -- all computation runs in the sm_100a
kernels under ``csrc/``.  PyTorch is used for device memory and streams only.
There is no CPU fallback: if the library is missing it is not silently
replaced, importing the compute entry points raises.
"""
from .binding import (  # noqa: F401
    FCFS, SJF, HRRN, DIST_LOGNORMAL, DIST_UNIFORM, REQ_DTYPE, SUMMARY_DTYPE, SPEC_DTYPE,
    REPLICA_DTYPE, COST_DTYPE, AsrSchedError, lib, lib_path, version, last_error, launch_count,
    workspace_bytes, to_device, tables_to_device, select, select_static, SELECT_STATIC_SCRATCH_BYTES, select_batched, simulate,
    simulate_batched, percentiles, gen_trace, gen_trace_batched, gen_queues, sweep_host,
    select_host, make_tables, make_replicas, make_cost, timing_enable, timing_reset, timing_read,
    set_option, OPT_SIM_LANE_MIN_REPLICAS, OPT_SIM_ESCALATE_WINDOW, OPT_SIM_LANE_SPLIT, ADAPTIVE, EXT_DTYPE, make_ext,
    simulate_batched_ex, tpot, estimate, itl_batched, trim_scratch,
)
