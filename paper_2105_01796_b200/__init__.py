"""paper_2105_01796_b200 -- B200-native batched Kalman-filter track fit (arxiv 2105.01796).

The product is the C-ABI library `libkf_fit.so` (include/kf_fit.h) built from `csrc/`;
`binding` marshals arguments into it; `workloads` generates the seeded synthetic inputs
(shared with the CPU oracle, and containing none of the fit's arithmetic).
"""
from . import workloads  # noqa: F401
from .binding import (DeviceBatch, DeviceOutputs, FitCall, HostBatch, HostCall, KfError,  # noqa: F401
                      fit_batch, fit_workload, lib, make_options, probe_fp64_tflops)
