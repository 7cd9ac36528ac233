"""dyplan: B200-native (sm_100a) hot path of Dyserve's physical-plan compiler (arxiv/paper_2607_02942).

``binding``   ctypes binding of the C ABI in include/dyplan.h (libdyplan.so, hand-written CUDA).
``workloads`` seeded synthetic inputs (numpy only; shared with the test oracle, holds no method arithmetic).
``build``     in-tree nvcc build of libdyplan.so.
"""
