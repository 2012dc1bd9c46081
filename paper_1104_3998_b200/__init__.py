"""pic1d -- B200-native 1D3V PIC/MCC hot path with per-cell fine sorting (arxiv 1104.3998).

`workloads` (seeded synthetic inputs, no method arithmetic) imports without CUDA; the
binding (`pic1d`) loads the CUDA C-ABI library lazily and fails loudly if it is missing.
"""
