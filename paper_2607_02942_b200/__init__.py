"""dyplan: B200-native (sm_100a) hot path of Dyserve's physical-plan compiler (arxiv/paper_2607_02942).

``binding``   ctypes binding of the C ABI in include/dyplan.h (libdyplan.so, hand-written CUDA).
``multi``     host logic of the N > 1 path (request sharding, max over ranks).
``cache``     host-side bundle cache.
``build``     in-tree nvcc build of libdyplan.so.
"""
