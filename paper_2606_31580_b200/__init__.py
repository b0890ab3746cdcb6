"""B200-native LASER confidence probe (arxiv/paper_2606_31580, §3.1 + §4.2 hot path).

`paper_2606_31580_b200.workloads` — seeded synthetic inputs (numpy only, importable anywhere).
`paper_2606_31580_b200.binding`   — thin ctypes binding of the C-ABI in include/laser_probe.h; every
                                    step of the path runs in the CUDA kernels of csrc/.  There is no
                                    CPU fallback: a missing library or a non-sm_100 device raises.
`paper_2606_31580_b200.build`     — nvcc build of csrc/ -> liblaser_probe.so (sm_100a only).
"""
__all__ = ["workloads", "binding", "build"]
