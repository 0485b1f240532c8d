"""psync: the parameter-server step of synchronous SGD with backup workers (arXiv 1702.05800,
Algorithm 4) as hand-written CUDA for sm_100a behind a C ABI (include/psync.h)."""
