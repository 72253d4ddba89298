"""B200-native time-reversible FDTD gradient loop with compressed boundary storage (arxiv/paper_2603_24027).

`paper_2603_24027_b200.fdtd` is the thin Python binding of the C-ABI library declared in include/fdtd.h
(hand-written sm_100a CUDA kernels under csrc/).  `paper_2603_24027_b200.workloads` holds the seeded
synthetic inputs.  Importing the package loads nothing native; the binding loads libfdtd_b200.so on first
use and raises if it is missing (there is no CPU fallback).
"""
