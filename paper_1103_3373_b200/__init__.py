"""B200-native unsplit hydro patch-group solver (arXiv:1103.3373 hot path).

`binding` holds the ctypes front end of the C ABI (include/hydro.h); `workloads` the seeded
synthetic inputs; `build` compiles csrc/ for sm_100a.  Nothing here imports oracle/.
"""
