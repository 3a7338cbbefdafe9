"""axg -- B200-native (sm_100a) axon-guidance time step: diffuse -> bin -> sense -> advance -> append.

`paper_1405_3331_b200.axg`       thin ctypes binding of the C-ABI library (include/axg.h)
`paper_1405_3331_b200.build`     nvcc build of csrc/ into libaxg.so (in-tree)
`paper_1405_3331_b200.workloads` seeded synthetic inputs C1..C5 (no arithmetic of the method)

Nothing here imports the CPU oracle; there is no CPU fallback.
"""
