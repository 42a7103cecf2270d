"""biobeam split-step BPM hot path, B200-native (sm_100a).  See DESIGN.md.

``binding`` wraps the C ABI of ``libbiobeam_b200.so`` (``include/bb.h``); ``workloads``
generates the seeded synthetic inputs; ``build`` compiles the library with nvcc.
"""
