"""B200-native (sm_100a) hot path of STREAmS-2 (arXiv 2304.05494): fused RHS + RK3 kernels
behind the C ABI of include/streams.h.  `binding` is the thin ctypes layer."""
